// slice_pipe_row.cu -- software-pipelined forms of the two slice-step passes (grids of 256 .. 2048).
//
// PAPER.md:44 Eq. (1)  psi <- psi * exp(i sigma V)          (transmission)
// PAPER.md:80 Eq. (2)  Psi <- Psi * exp(-i pi lambda q^2 t)  (propagation), "done in Fourier space"
//
// Same arithmetic and the same two-pass structure as slice_pass.cu (row pass IFFT_x . t . FFT_x,
// column pass FFT_y . P . IFFT_y, wave kept in mixed space A[w][y][kx] between them), organised so
// that HBM transfers, shared-memory exchanges and butterflies of different lines overlap:
//
//  * every thread holds E = 32 points, so lines up to 1024 points need ONE shared-memory exchange
//    per transform (2048: two) and inter-stage twiddles come from a transposed shared table;
//  * row pass: a team (one warp; two for 2048-point lines) owns a private two-slot ring that the
//    TMA engine fills with 1-D bulk copies (cp.async.bulk + mbarrier transaction counts); the slot
//    the line lands in is also its exchange space; results go straight from registers to HBM.
//    There is no CTA-wide barrier in the loop;
//  * column pass: two teams of 256 threads per CTA alternate over [N rows] x [W columns] tiles of
//    8192 points held in a three-buffer ring filled by 16-byte cp.async copies that signal an
//    mbarrier; a lane owns one column of the tile and consecutive lanes consecutive columns, so every
//    shared-memory access of the transforms is a contiguous run and results are stored from
//    registers as 64-byte (W = 8) row segments;
//  * band-limit: after the column pass everything with |kx| > kx_max is exactly zero (2/3 rule,
//    BASELINE.json), so mixed space is only ever read and written for kx in [0, xband) and
//    [nx - xband, nx): the column pass runs on 2 xband / W tiles per wave and the row pass moves
//    2 xband of the nx points of a line.
// complex adds of the register butterflies as packed FADD2 (measured: 3-7 % faster row pass, slower column pass)
#define PRISM_PACKED_ADDS 1
#include "fft_core.cuh"
#include "pipe_plan.cuh"
#include "prism_internal.h"
#include "pipe_ptx.cuh"

namespace prism {

// =============================================================================
// Row pass
// =============================================================================
template <class P>
struct RowCfg {
    static constexpr int T = P::T;
    static constexpr int TEAM = T < 32 ? 32 : T;                 // threads of one team
    static constexpr int LPT = TEAM / T;                         // lines per team
    static constexpr int LINE = P::N + 2 * (P::N / P::R1);       // padded exchange space of one line (float2)
    static constexpr int SLOT = LPT * LINE;
    static constexpr int TWB = round_up_c(SmemTwiddles<P>::COUNT * 8, 128);
    static constexpr int TEAMS_BY_SMEM = (PIPE_SMEM_MAX - PIPE_HEADER - TWB) / (2 * SLOT * 8);
    static constexpr int TEAMS = TEAMS_BY_SMEM < 384 / TEAM ? TEAMS_BY_SMEM : 384 / TEAM;
    static constexpr int THREADS = TEAMS * TEAM;
    static constexpr size_t SMEM = PIPE_HEADER + TWB + (size_t)TEAMS * 2 * SLOT * 8;
};

// exchange space of one line inside its slot: element idx at base[idx + 2 (idx / R1)].  Two pad words per
// group of R1 keep pairs (even idx, idx + 1) 16-byte aligned, so the radix-R1 outputs of a thread go out as
// 16-byte stores, and a quarter warp of such stores (stride R1 + 2 words) covers all banks once.
template <class P, int TEAM>
struct RowSm {
    float2* base;
    int bar_id;
    __device__ __forceinline__ static int phys(int idx) { return idx + 2 * (idx / P::R1); }
    __device__ __forceinline__ void  st(int idx, float2 v) const { base[phys(idx)] = v; }
    __device__ __forceinline__ void  st2(int idx, float2 v0, float2 v1) const
    { *reinterpret_cast<float4*>(base + phys(idx)) = make_float4(v0.x, v0.y, v1.x, v1.y); }
    __device__ __forceinline__ float2 ld(int idx) const { return base[phys(idx)]; }
    __device__ __forceinline__ void sync() const { if (TEAM <= 32) __syncwarp(); else named_barrier(bar_id, TEAM); }
};

// XBE > 0: the band is xband = XBE * T columns, known at compile time (then "in band" depends on the register
// index e only and out-of-band elements cost no instruction); XBE = 0: any xband, tested per element.
template <class P, int MODE, int XBE>
__global__ void __launch_bounds__(RowCfg<P>::THREADS, 1) row_pipe_kernel(RowArgs g)
{
    using C = RowCfg<P>;
    constexpr int E = P::E, T = P::T, N = P::N;
    auto in_band = [&](int e, int kx, int xb) { return XBE > 0 ? (e < XBE || e >= E - XBE) : (kx < xb || kx >= N - xb); };
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw);                    // [TEAMS][2]
    float2* twtab = reinterpret_cast<float2*>(smem_raw + PIPE_HEADER);
    float2* slots = reinterpret_cast<float2*>(smem_raw + PIPE_HEADER + C::TWB);
    const int tid = threadIdx.x, team = tid / C::TEAM, tt = tid % C::TEAM;
    const int ll = tt / T, t = tt % T;

    SmemTwiddles<P>::fill(twtab, g.tw_x, tid, C::THREADS);
    if (MODE != ROW_INIT && tt == 0) {
        mbar_init(&bars[team * 2], 1);
        mbar_init(&bars[team * 2 + 1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    SmemTwiddles<P> tw;
    tw.bind(twtab, t);
    float2* slot0 = slots + (size_t)team * 2 * C::SLOT;

    const long long n_lines = (long long)g.n_waves * g.ny;
    const long long n_groups = (n_lines + C::LPT - 1) / C::LPT;
    const long long gteam = (long long)blockIdx.x * C::TEAMS + team, gstride = (long long)gridDim.x * C::TEAMS;
    const int xb = XBE > 0 ? XBE * T : g.xband;              // in-band columns: [0, xb) and [N - xb, N)

    // one thread of the team: start the bulk copies of line group `grp` into slot `s`
    auto issue = [&](long long grp, int s) {
        uint64_t* bar = &bars[team * 2 + s];
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
                float2* dst = slot0 + s * C::SLOT + l * C::LINE;
                bulk_g2s(dst, row, (unsigned)(xb * sizeof(float2)), bar);
                bulk_g2s(dst + (N - xb), row + (N - xb), (unsigned)(xb * sizeof(float2)), bar);
            }
        }
    };
    if (MODE != ROW_INIT && tt == 0) {
        if (gteam < n_groups) issue(gteam, 0);
        if (gteam + gstride < n_groups) issue(gteam + gstride, 1);
    }

    int it = 0;
    for (long long grp = gteam; grp < n_groups; grp += gstride, ++it) {
        const int s = it & 1;
        long long line = grp * C::LPT + ll;
        const bool active = line < n_lines;
        if (!active) line = n_lines - 1;                 // keep every thread in the barriers
        const int y = (int)(line / g.n_waves), w = (int)(line % g.n_waves);
        float2* row = g.a + ((size_t)w * g.ny + y) * N;
        float2* lbase = slot0 + s * C::SLOT + ll * C::LINE;
        const RowSm<P, C::TEAM> sm{ lbase, 1 + team };
        float2 v[E];

        if (MODE == ROW_INIT) {
            // plane wave exp(+2 pi i (kx x / nx + ky y / ny)) * amplitude
            const int2 b = g.beams[w];
            const float2 wy = __ldg(g.tw_y + ((b.y * y) & (g.ny - 1)));
            const float2 base = make_float2(wy.x * g.scale, -wy.y * g.scale);
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const float2 wx = __ldg(g.tw_x + ((b.x * (t + T * e)) & (N - 1)));
                v[e] = cmul_conj(base, wx);
            }
        } else {
            mbar_wait(&bars[team * 2 + s], (unsigned)((it >> 1) & 1));
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const int kx = t + T * e;
                v[e] = in_band(e, kx, xb) ? lbase[kx] : make_float2(0.f, 0.f);   // out of band: exact zeros
            }
        }

        if (MODE == ROW_STEP || MODE == ROW_FINAL) fft_inverse<P>(v, tw, t, sm);

        if (MODE == ROW_INIT || MODE == ROW_STEP) {
            const float2* trow = g.t + (size_t)y * N;
#pragma unroll
            for (int e = 0; e < E; ++e) v[e] = cmul(v[e], __ldg(trow + t + T * e));
        }
        if (MODE != ROW_FINAL) fft_forward<P>(v, tw, t, sm);

        if (MODE != ROW_INIT) {
            // the slot is free once every thread of the team is past its last exchange read
            sm.sync();
            if (tt == 0) {
                const long long nxt = grp + 2 * gstride;
                if (nxt < n_groups) { fence_proxy_async(); issue(nxt, s); }
            }
        }

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
    using C = RowCfg<P>;
    auto kern = row_pipe_kernel<P, MODE, XBE>;
    static bool set = false;
    if (!set) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
        if (e != cudaSuccess) return e;
        set = true;
    }
    const long long n_lines = (long long)g.n_waves * g.ny;
    const long long n_groups = (n_lines + C::LPT - 1) / C::LPT;
    if (n_groups == 0) return cudaSuccess;
    long long grid = (n_groups + C::TEAMS - 1) / C::TEAMS;
    if (grid > num_sms()) grid = num_sms();
    kern<<<(unsigned)grid, C::THREADS, C::SMEM, stream>>>(g);
    return cudaGetLastError();
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
        case 2048: return launch_row_pipe_n<2048>(mode, g, stream);
    }
    return cudaErrorInvalidValue;
}

}  // namespace prism
