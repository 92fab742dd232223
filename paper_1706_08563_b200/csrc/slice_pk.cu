// slice_pk.cu -- slice-step passes on the two-way packed FFT of fft_pk.cuh (FADD2 / FMUL2 / FFMA2).
//
// PAPER.md:44 Eq. (1)  psi <- psi * exp(i sigma V)          (transmission)
// PAPER.md:80 Eq. (2)  Psi <- Psi * exp(-i pi lambda q^2 t)  (propagation), "done in Fourier space"
//
// Same two passes, same mixed-space storage A[w][y][kx] and the same band-limit bookkeeping as
// slice_pipe_row.cu / slice_pipe_col.cu; what changes is the transform: a line of N points is held by N / 64 threads (64 points
// each), split by one radix-2 step in registers into two half-length transforms that run as the two
// lanes of packed fp32 instructions, so a transform needs ONE shared-memory exchange up to 2048 points,
// only warp-level barriers in the row pass, and about half the instructions per point:
//
//   row pass    : A (natural kx) -> inverse DIF -> real space in pairs (x[2j], x[2j+1]) -> * t_s (stored in
//                 the same pair layout by the transmission kernel) -> forward DIT -> A (natural kx)
//   column pass : A (natural y) -> forward DIF -> pairs (ky = 2j, 2j+1) -> * P -> inverse DIT -> A (natural y)
//
// so global memory is always read and written in natural order with coalesced accesses and no register
// shuffling is needed between the pair layout and memory.
//
// Blocked mixed space "B8" (square 2048-point grids; prism_internal.h `blocked_grid`): between the two passes a
// wave holds only its 2 xb in-band columns, in compact order j (j < xb: kx = j; j >= xb: slot nx - 2 xb + j), as
// tiles of 8 columns,   element (y, j) at  a[w nx ny + ((j >> 3) ny + y) 8 + (j & 7)],
// so that a column tile [ny rows] x [8 columns] is ONE contiguous 128 KB run: the column pass fetches it with a
// few bulk copies (no LSU work) and stores it back from registers as 256-byte runs (4 rows x 64 B per warp
// instruction) instead of 32-byte row segments; the row pass gathers a line as 2 xb / 8 pieces of 64 bytes
// (one 4-D TMA tensor box, or 16-byte cp.async copies) and stores 4 x 64 B per warp instruction.
#include <cuda.h>

#include "fft_core.cuh"
#include "fft_pk.cuh"
#include "pipe_ptx.cuh"
#include "prism_internal.h"

#include <atomic>
#include <cstring>

namespace prism {

using pk::C2;

constexpr int PK_ROW_MAX_WARPS = 8;

// =============================================================================
// Row pass
// =============================================================================
// XBE < 32: the band is xband = XBE * T columns, known at compile time; XBE = 32: any xband, tested per element.
template <int N, int XBE>
struct RowPkCfg {
    using P = pk::PkPlan<N>;
    static constexpr int T = P::T, LPW = 32 / T;                   // threads per line, lines per warp
    static constexpr int LANDW = XBE < 32 ? 2 * XBE * T : N;       // points of a line that are moved
    static constexpr int LAND_BYTES = LPW * LANDW * 8;
    static constexpr int X_BYTES = LPW * P::XPAD * 8;               // one 8-byte plane, used in two phases
    static constexpr int PER_WARP = LAND_BYTES + X_BYTES;
    static constexpr int TWB = round_up_c(P::TW_BYTES, 128);
    static constexpr int BY_SMEM = (PIPE_SMEM_MAX - PIPE_HEADER - TWB) / PER_WARP;
    static constexpr int WARPS = BY_SMEM < PK_ROW_MAX_WARPS ? BY_SMEM : PK_ROW_MAX_WARPS;
    static constexpr int THREADS = WARPS * 32;
    static constexpr size_t SMEM = PIPE_HEADER + TWB + (size_t)WARPS * PER_WARP;
};

template <int N, int MODE, int XBE>
__global__ void __launch_bounds__(RowPkCfg<N, XBE>::THREADS, 1) row_pk_kernel(RowArgs g)
{
    using C = RowPkCfg<N, XBE>;
    using P = typename C::P;
    constexpr int T = P::T, LPW = C::LPW;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw);                    // [WARPS]
    float2* tab = reinterpret_cast<float2*>(smem_raw + PIPE_HEADER);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int ll = lane / T, t = lane % T;
    unsigned char* mine = smem_raw + PIPE_HEADER + C::TWB + (size_t)warp * C::PER_WARP;
    float2* land = reinterpret_cast<float2*>(mine);                            // [LPW][LANDW]
    float2* xch = reinterpret_cast<float2*>(mine + C::LAND_BYTES);             // [LPW][XPAD]

    pk::fill_tables<P>(tab, g.tw_x, tid, C::THREADS);
    if (MODE != ROW_INIT && lane == 0) { mbar_init(&bars[warp], 1); mbar_fence_init(); }
    __syncthreads();
    griddep_wait();                          // the previous kernel of the slice loop has completed (pipe_ptx.cuh)

    const long long n_lines = (long long)g.n_waves * g.ny;
    const long long n_groups = (n_lines + LPW - 1) / LPW;
    const long long gw = (long long)blockIdx.x * C::WARPS + warp, gstride = (long long)gridDim.x * C::WARPS;
    const int xb = XBE < 32 ? XBE * T : g.xband;                 // in-band columns: [0, xb) and [N - xb, N)

    // lane 0: start the bulk copies of line group `grp` into the landing buffer
    auto issue = [&](long long grp) {
        int n_act = 0;
#pragma unroll
        for (int l = 0; l < LPW; ++l) n_act += (grp * LPW + l < n_lines);
        mbar_expect_tx(&bars[warp], (unsigned)(n_act * 2 * xb * (int)sizeof(float2)));
#pragma unroll
        for (int l = 0; l < LPW; ++l) {
            const long long line = grp * LPW + l;
            if (line < n_lines) {
                const int y = (int)(line / g.n_waves), w = (int)(line % g.n_waves);
                const float2* row = g.a + ((size_t)w * g.ny + y) * N;
                float2* dst = land + l * C::LANDW;
                bulk_g2s(dst, row, (unsigned)(xb * sizeof(float2)), &bars[warp]);
                bulk_g2s(dst + xb, row + (N - xb), (unsigned)(xb * sizeof(float2)), &bars[warp]);
            }
        }
    };
    if (MODE != ROW_INIT && lane == 0 && gw < n_groups) issue(gw);

    const pk::XchgPhase sm{ xch + ll * P::XPAD, 1 };
    auto sync = [] { __syncwarp(); };
    auto in_band = [&](int e) { return XBE < 32 ? pk::kept<XBE>(e) : (t + T * e < xb || t + T * e >= N - xb); };

    int it = 0;
    for (long long grp = gw; grp < n_groups; grp += gstride, ++it) {
        long long line = grp * LPW + ll;
        const bool active = line < n_lines;
        if (!active) line = n_lines - 1;                 // keep every lane in the warp barriers
        const int y = (int)(line / g.n_waves), w = (int)(line % g.n_waves);
        float2* row = g.a + ((size_t)w * g.ny + y) * N;
        C2 p[32];

        // Phase 0 builds the pairs the first half-length transform runs on (plane wave, or the landed line after
        // the radix-2 step of the inverse DIF); phase 1 multiplies by t_s between the inverse and the forward
        // transform.  ROW_STEP runs both phases through ONE copy of the transform code (instruction cache).
        constexpr int PH0 = (MODE == ROW_INIT) ? 1 : 0, PH1 = (MODE == ROW_FINAL) ? 1 : 2;
#pragma unroll 1
        for (int ph = PH0; ph < PH1; ++ph) {
            if (ph == 0) {
                float2 v[64];
                mbar_wait(&bars[warp], (unsigned)(it & 1));
                const float2* lbase = land + ll * C::LANDW;
#pragma unroll
                for (int e = 0; e < 64; ++e) {
                    const int kx = t + T * e;
                    int pos;                                    // compact landing: [0, xb) then [N - xb, N)
                    if (XBE < 32) pos = e < XBE ? kx : kx - (N - 2 * xb);
                    else pos = kx < xb ? kx : (kx >= N - xb ? kx - (N - 2 * xb) : 0);
                    if (XBE < 32 && !pk::kept<XBE>(e)) { v[e] = make_float2(0.f, 0.f); continue; }
                    const float2 q = lbase[pos];
                    v[e] = in_band(e) ? make_float2(q.y, q.x) : make_float2(0.f, 0.f);   // (im, re): inverse = swapped forward
                }
                // the landing buffer is free once every lane has read its points
                __syncwarp();
                if (lane == 0 && grp + gstride < n_groups) { fence_proxy_async(); issue(grp + gstride); }
                pk::dif_pre<P, XBE>(v, p, tab, t);
            } else {
                if (MODE == ROW_INIT) {
                    // plane wave exp(+2 pi i (kx x / nx + ky y / ny)) * amplitude at x = 2 j, 2 j + 1
                    const int2 b = g.beams[w];
                    const float2 wy = __ldg(g.tw_y + ((b.y * y) & (g.ny - 1)));
                    const float2 base = make_float2(wy.x * g.scale, -wy.y * g.scale);
                    // x = 2 (t + T e) + {0, 1}: one gathered table value per thread and parity, one warp-uniform
                    // value per slot (conj(w^(kx x)) = conj(w^(kx (2 t + h))) conj(w^(kx 2 T e)))
                    const float2 b0 = cmul_conj(base, __ldg(g.tw_x + ((b.x * (2 * t)) & (N - 1))));
                    const float2 b1 = cmul_conj(base, __ldg(g.tw_x + ((b.x * (2 * t + 1)) & (N - 1))));
#pragma unroll
                    for (int e = 0; e < 32; ++e) {
                        const float2 we = __ldg(g.tw_x + ((b.x * (2 * T * e)) & (N - 1)));
                        const float2 v0 = cmul_conj(b0, we), v1 = cmul_conj(b1, we);
                        p[e] = { make_float2(v0.x, v1.x), make_float2(v0.y, v1.y) };
                    }
                } else {
#pragma unroll
                    for (int e = 0; e < 32; ++e) p[e] = pk::cswap(p[e]);       // back from the swapped inverse
                }
                // transmission function in pair layout: (re(2j), re(2j+1), im(2j), im(2j+1))
                const float4* trow = reinterpret_cast<const float4*>(g.t) + (size_t)y * (N / 2);
#pragma unroll
                for (int e = 0; e < 32; ++e) {
                    const float4 q = __ldg(trow + t + T * e);
                    p[e] = pk::cmul2(p[e], make_float2(q.x, q.y), make_float2(q.z, q.w));
                }
            }
            pk::fft_half<P>(p, tab, t, sm, sync);
        }

        if (MODE == ROW_FINAL) {
            float4* dst = reinterpret_cast<float4*>(g.out + ((size_t)w * g.ny + y) * N);
            if (active) {
#pragma unroll
                for (int e = 0; e < 32; ++e)       // p holds the swapped inverse: (y, x) are (re, im)
                    dst[t + T * e] = make_float4(p[e].y.x * g.scale, p[e].x.x * g.scale, p[e].y.y * g.scale, p[e].x.y * g.scale);
            }
        } else {
            float2 v[64];
            pk::dit_post<P, XBE>(p, v, tab, t);
            if (active) {
#pragma unroll
                for (int e = 0; e < 64; ++e)
                    if (in_band(e)) row[t + T * e] = v[e];
            }
        }
    }
}

template <int N, int MODE, int XBE>
static cudaError_t launch_row_pk_x(const RowArgs& g, cudaStream_t stream)
{
    using C = RowPkCfg<N, XBE>;
    auto kern = row_pk_kernel<N, MODE, XBE>;
    static PerDevice once{};
    if (cudaError_t e = opt_in_smem(kern, C::SMEM, once); e != cudaSuccess) return e;
    const long long n_lines = (long long)g.n_waves * g.ny;
    const long long n_groups = (n_lines + C::LPW - 1) / C::LPW;
    if (n_groups == 0) return cudaSuccess;
    long long grid = (n_groups + C::WARPS - 1) / C::WARPS;
    if (grid > num_sms()) grid = num_sms();
    return launch_pdl(kern, (unsigned)grid, C::THREADS, C::SMEM, stream, g);
}

template <int N, int MODE>
static cudaError_t launch_row_pk_t(const RowArgs& g, cudaStream_t stream)
{
    constexpr int XB = DefaultBand<N>::XB, T = N / 64;
    static_assert(XB % T == 0, "default band must be a whole number of register slots");
    if (g.xband == XB) return launch_row_pk_x<N, MODE, XB / T>(g, stream);
    return launch_row_pk_x<N, MODE, 32>(g, stream);
}

template <int N>
static cudaError_t launch_row_pk_n(RowMode mode, const RowArgs& g, cudaStream_t stream)
{
    switch (mode) {
        case ROW_INIT:  return launch_row_pk_t<N, ROW_INIT>(g, stream);
        case ROW_STEP:  return launch_row_pk_t<N, ROW_STEP>(g, stream);
        case ROW_FINAL: return launch_row_pk_t<N, ROW_FINAL>(g, stream);
        default: break;
    }
    return cudaErrorInvalidValue;
}

template <int N> static cudaError_t launch_row_b8(RowMode mode, const RowArgs& g, cudaStream_t stream);   // below

cudaError_t launch_row_pk(RowMode mode, const RowArgs& g, cudaStream_t stream)
{
    if (g.xband < 32 || g.xband % 32 || 2 * g.xband > g.nx) return cudaErrorInvalidValue;
    if (g.blocked) return g.nx == 2048 ? launch_row_b8<2048>(mode, g, stream) : cudaErrorInvalidValue;
    switch (g.nx) {
        case 1024: return launch_row_pk_n<1024>(mode, g, stream);
        case 2048: return launch_row_pk_n<2048>(mode, g, stream);
    }
    return cudaErrorInvalidValue;
}

// =============================================================================
// Row pass on the blocked layout "B8" (top of this file)
// =============================================================================
// A line of blocked mixed space is 2 xb / 8 pieces of 64 bytes, 128 KB apart; pieces of consecutive rows y are
// adjacent.  So that the DRAM sees runs and not isolated 64-byte pieces, lines are ordered by (block of G rows,
// group of 8 waves): CTA b of the G resident CTAs owns row y = yb G + b of the current row block and its 8 warps
// take 8 different waves of that row -- at any moment the grid reads and writes G consecutive rows of a few waves,
// i.e. runs of G x 64 B per tile.  Every warp of a CTA then needs the same row of the transmission function for
// n_waves / 8 lines in a row: it is brought into shared memory once per row block (one bulk copy), which takes the
// t_s loads out of the L1 / long-scoreboard path.
// The line is gathered by one 4-D TMA tensor box {8 columns, 1 row, 2 xb / 8 tiles, 1 wave} issued by one lane
// (16-byte cp.async copies by all lanes were measured slower: DESIGN.md 7.8).
__device__ __forceinline__ void tensor_g2s_4d(void* smem_dst, const CUtensorMap* map, int c0, int c1, int c2, int c3,
                                              uint64_t* bar)
{
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                 ::"r"(smem_u32(smem_dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)) : "memory");
}

template <int N, int XBE>
struct RowB8Cfg {
    using P = pk::PkPlan<N>;
    using B = RowPkCfg<N, XBE>;
    static constexpr int T = P::T, LPW = 32 / T;
    static constexpr int LANDW = B::LANDW, LAND_BYTES = B::LAND_BYTES, PER_WARP = B::PER_WARP, TWB = B::TWB;
    static constexpr int T_BYTES = N * 8;                          // one row of the transmission function
    static constexpr int BY_SMEM = (PIPE_SMEM_MAX - PIPE_HEADER - TWB - T_BYTES) / PER_WARP;
    static constexpr int WARPS = BY_SMEM < PK_ROW_MAX_WARPS ? BY_SMEM : PK_ROW_MAX_WARPS;
    static constexpr int THREADS = WARPS * 32;
    static constexpr size_t SMEM = PIPE_HEADER + TWB + T_BYTES + (size_t)WARPS * PER_WARP;
};

template <int N, int MODE, int XBE>
__global__ void __launch_bounds__(RowB8Cfg<N, XBE>::THREADS, 1) row_b8_kernel(RowArgs g, const __grid_constant__ CUtensorMap tmap)
{
    using C = RowB8Cfg<N, XBE>;
    using P = typename C::P;
    constexpr int T = P::T, LPW = C::LPW, WARPS = C::WARPS;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw);                    // [WARPS] landing buffers, [WARPS] t row
    float2* tab = reinterpret_cast<float2*>(smem_raw + PIPE_HEADER);
    const float4* trow = reinterpret_cast<const float4*>(smem_raw + PIPE_HEADER + C::TWB);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int ll = lane / T, t = lane % T;
    unsigned char* mine = smem_raw + PIPE_HEADER + C::TWB + C::T_BYTES + (size_t)warp * C::PER_WARP;
    float2* land = reinterpret_cast<float2*>(mine);                            // [LPW][LANDW]
    float2* xch = reinterpret_cast<float2*>(mine + C::LAND_BYTES);             // [LPW][XPAD]
    uint64_t* tbar = &bars[WARPS];

    pk::fill_tables<P>(tab, g.tw_x, tid, C::THREADS);
    if (lane == 0) {
        if (MODE != ROW_INIT) mbar_init(&bars[warp], 1);
        if (warp == 0) mbar_init(tbar, 1);
        mbar_fence_init();
    }
    __syncthreads();
    griddep_wait();                          // the previous kernel of the slice loop has completed (pipe_ptx.cuh)

    const int G = gridDim.x, bid = blockIdx.x;
    constexpr size_t wave_stride = (size_t)N * N;                 // blocked grids are square: ny == N
    const int xb = XBE < 32 ? XBE * T : g.xband;                 // in-band columns: [0, xb) and [N - xb, N)
    // this warp's lines: rows y = yb G + bid (yb < my_yblocks), wave groups wg < my_wgroups with waves
    // (wg WARPS + warp) LPW + l; `seq` = yb my_wgroups + wg numbers them in processing order
    const int my_yblocks = bid < g.ny ? (g.ny - bid + G - 1) / G : 0;
    const int first_wave = warp * LPW;
    const int my_wgroups = first_wave < g.n_waves ? (g.n_waves - first_wave + WARPS * LPW - 1) / (WARPS * LPW) : 0;
    const long long my_lines = (long long)my_yblocks * my_wgroups;

    // start the copies of line group `seq` into the landing buffer (compact: [0, xb) then [N - xb, N)).
    // Called by lane 0.
    auto issue = [&](long long seq) {
        const int y = (int)(seq / my_wgroups) * G + bid, w0 = ((int)(seq % my_wgroups) * WARPS + warp) * LPW;
        int n_act = 0;
#pragma unroll
        for (int l = 0; l < LPW; ++l) n_act += (w0 + l < g.n_waves);
        mbar_expect_tx(&bars[warp], (unsigned)(n_act * 2 * xb * (int)sizeof(float2)));
#pragma unroll
        for (int l = 0; l < LPW; ++l)
            if (w0 + l < g.n_waves) tensor_g2s_4d(land + l * C::LANDW, &tmap, 0, y, 0, w0 + l, &bars[warp]);
    };
    if (MODE != ROW_INIT && lane == 0 && my_lines > 0) issue(0);

    const pk::XchgPhase sm{ xch + ll * P::XPAD, 1 };
    auto sync = [] { __syncwarp(); };
    auto in_band = [&](int e) { return XBE < 32 ? pk::kept<XBE>(e) : (t + T * e < xb || t + T * e >= N - xb); };

    long long seq = 0;
    for (int yb = 0; yb < my_yblocks; ++yb) {
        const int y = yb * G + bid;
        if (MODE != ROW_FINAL) {
            // the row of t_s every warp of this CTA multiplies by until the next row block
            __syncthreads();                             // every warp is done with the previous row
            if (tid == 0) {
                fence_proxy_async();
                mbar_expect_tx(tbar, (unsigned)C::T_BYTES);
                bulk_g2s(const_cast<float4*>(trow), g.t + (size_t)y * N, (unsigned)C::T_BYTES, tbar);
            }
            mbar_wait(tbar, (unsigned)(yb & 1));
        }
        for (int wg = 0; wg < my_wgroups; ++wg, ++seq) {
            int w = (wg * WARPS + warp) * LPW + ll;
            const bool active = w < g.n_waves;
            if (!active) w = g.n_waves - 1;                  // keep every lane in the warp barriers
            // row y of tile 0 of the wave; column j of the compact band lives (j >> 3) ny 8 + (j & 7) further on
            float2* row = g.a + (size_t)w * wave_stride + (size_t)y * 8;
            C2 p[32];

            constexpr int PH0 = (MODE == ROW_INIT) ? 1 : 0, PH1 = (MODE == ROW_FINAL) ? 1 : 2;
#pragma unroll 1
            for (int ph = PH0; ph < PH1; ++ph) {
                if (ph == 0) {
                    float2 v[64];
                    mbar_wait(&bars[warp], (unsigned)(seq & 1));
                    const float2* lbase = land + ll * C::LANDW;
#pragma unroll
                    for (int e = 0; e < 64; ++e) {
                        const int kx = t + T * e;
                        int pos;                                    // compact landing: [0, xb) then [N - xb, N)
                        if (XBE < 32) pos = e < XBE ? kx : kx - (N - 2 * xb);
                        else pos = kx < xb ? kx : (kx >= N - xb ? kx - (N - 2 * xb) : 0);
                        if (XBE < 32 && !pk::kept<XBE>(e)) { v[e] = make_float2(0.f, 0.f); continue; }
                        const float2 q = lbase[pos];
                        v[e] = in_band(e) ? q : make_float2(0.f, 0.f);
                    }
                    // the landing buffer is free once every lane has read its points
                    __syncwarp();
                    if (seq + 1 < my_lines && lane == 0) { fence_proxy_async(); issue(seq + 1); }
                    pk::dif_pre<P, XBE, true>(v, p, tab, t);       // inverse = conj of the forward transform of conj(v)
                } else {
                    if (MODE == ROW_INIT) {
                        // plane wave exp(+2 pi i (kx x / nx + ky y / ny)) * amplitude at x = 2 j, 2 j + 1
                        const int2 b = g.beams[w];
                        const float2 wy = __ldg(g.tw_y + ((b.y * y) & (g.ny - 1)));
                        const float2 base = make_float2(wy.x * g.scale, -wy.y * g.scale);
                        const float2 b0 = cmul_conj(base, __ldg(g.tw_x + ((b.x * (2 * t)) & (N - 1))));
                        const float2 b1 = cmul_conj(base, __ldg(g.tw_x + ((b.x * (2 * t + 1)) & (N - 1))));
#pragma unroll
                        for (int e = 0; e < 32; ++e) {
                            const float2 we = __ldg(g.tw_x + ((b.x * (2 * T * e)) & (N - 1)));
                            const float2 v0 = cmul_conj(b0, we), v1 = cmul_conj(b1, we);
                            p[e] = { make_float2(v0.x, v1.x), make_float2(v0.y, v1.y) };
                        }
                    }
                    // transmission function in pair layout: (re(2j), re(2j+1), im(2j), im(2j+1)); after the inverse p
                    // holds the conjugate of the real-space line
#pragma unroll
                    for (int e = 0; e < 32; ++e) {
                        const float4 q = trow[t + T * e];
                        if (MODE == ROW_INIT) p[e] = pk::cmul2(p[e], make_float2(q.x, q.y), make_float2(q.z, q.w));
                        else p[e] = pk::cmul2_conj(p[e], make_float2(q.x, q.y), make_float2(q.z, q.w));
                    }
                }
                pk::fft_half<P>(p, tab, t, sm, sync);
            }

            if (MODE == ROW_FINAL) {
                float4* dst = reinterpret_cast<float4*>(g.out + ((size_t)w * g.ny + y) * N);
                if (active) {
#pragma unroll
                    for (int e = 0; e < 32; ++e)       // p holds the conjugate of the inverse
                        dst[t + T * e] = make_float4(p[e].x.x * g.scale, -p[e].y.x * g.scale, p[e].x.y * g.scale, -p[e].y.y * g.scale);
                }
            } else {
                float2 v[64];
                pk::dit_post<P, XBE>(p, v, tab, t);
                if (active) {
                    // compact column j = t + T e' (e' = e below the gap, e - gap above it) sits (j >> 3) tiles further
                    // on: with T = 32 that is 4 e' tiles of N x 8 points, a compile-time stride per register slot
                    static_assert(T % 8 == 0, "tile arithmetic");
                    float2* rowt = row + (size_t)(t >> 3) * N * 8 + (t & 7);
#pragma unroll
                    for (int e = 0; e < 64; ++e) {
                        if (!in_band(e)) continue;
                        if (XBE < 32) {
                            const int ep = e < XBE ? e : e - (64 - 2 * XBE);
                            rowt[(size_t)ep * (T / 8) * N * 8] = v[e];
                        } else {
                            const int kx = t + T * e;
                            const int j = kx < xb ? kx : kx - (N - 2 * xb);
                            row[(size_t)(j >> 3) * N * 8 + (j & 7)] = v[e];
                        }
                    }
                }
            }
        }
    }
}

// 4-D tensor map over the blocked mixed space of a wave batch: dims (fastest first) {16 floats = 8 columns, ny rows,
// 2 xb / 8 tiles, n_waves}; the box {16, 1, 2 xb / 8, 1} is one compact line.  The driver entry point is fetched at
// run time (no link-time dependency on libcuda).
static cudaError_t encode_line_map(const RowArgs& g, CUtensorMap* map)
{
    typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static std::atomic<void*> cached{nullptr};
    void* fn = cached.load(std::memory_order_acquire);
    if (!fn) {
        cudaDriverEntryPointQueryResult qres;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
        if (e != cudaSuccess) return e;
        if (!fn || qres != cudaDriverEntryPointSuccess) return cudaErrorNotSupported;
        cached.store(fn, std::memory_order_release);
    }
    const cuuint64_t tiles = (cuuint64_t)(2 * g.xband / 8);
    if (tiles > 256) return cudaErrorInvalidValue;
    const cuuint64_t dims[4] = { 16, (cuuint64_t)g.ny, tiles, (cuuint64_t)g.n_waves };
    const cuuint64_t strides[3] = { 64, (cuuint64_t)g.ny * 64, (cuuint64_t)g.nx * g.ny * 8 };
    const cuuint32_t box[4] = { 16, 1, (cuuint32_t)tiles, 1 };
    const cuuint32_t estr[4] = { 1, 1, 1, 1 };
    const CUresult r = ((EncodeFn)fn)(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, (void*)g.a, dims, strides, box, estr,
                                      CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                      CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

template <int N, int MODE, int XBE>
static cudaError_t launch_row_b8_x(const RowArgs& g, cudaStream_t stream)
{
    using C = RowB8Cfg<N, XBE>;
    auto kern = row_b8_kernel<N, MODE, XBE>;
    static PerDevice once{};
    if (cudaError_t e = opt_in_smem(kern, C::SMEM, once); e != cudaSuccess) return e;
    if (g.n_waves <= 0) return cudaSuccess;
    if (g.ny != N) return cudaErrorInvalidValue;                                  // blocked grids are square
    if (MODE == ROW_FINAL && g.out == g.a) return cudaErrorInvalidValue;          // the layouts differ: not in place
    int grid = num_sms();
    if (grid > g.ny) grid = g.ny;
    CUtensorMap map;
    std::memset(&map, 0, sizeof(map));
    if (MODE != ROW_INIT)
        if (cudaError_t e = encode_line_map(g, &map); e != cudaSuccess) return e;
    return launch_pdl(kern, (unsigned)grid, C::THREADS, C::SMEM, stream, g, map);
}

template <int N>
static cudaError_t launch_row_b8(RowMode mode, const RowArgs& g, cudaStream_t stream)
{
    constexpr int XB = DefaultBand<N>::XB, T = N / 64;
    const bool def = g.xband == XB;
    switch (mode) {
        case ROW_INIT:  return def ? launch_row_b8_x<N, ROW_INIT, XB / T>(g, stream) : launch_row_b8_x<N, ROW_INIT, 32>(g, stream);
        case ROW_STEP:  return def ? launch_row_b8_x<N, ROW_STEP, XB / T>(g, stream) : launch_row_b8_x<N, ROW_STEP, 32>(g, stream);
        case ROW_FINAL: return def ? launch_row_b8_x<N, ROW_FINAL, XB / T>(g, stream) : launch_row_b8_x<N, ROW_FINAL, 32>(g, stream);
        default: break;
    }
    return cudaErrorInvalidValue;
}

// =============================================================================
// Column pass
// =============================================================================
template <int N>
struct ColPkCfg {
    using P = pk::PkPlan<N>;
    static constexpr int T = P::T;
    static constexpr int TILE_PTS = 8192;
    static constexpr int W = TILE_PTS / N;                       // columns per tile: 8 (1024), 4 (2048)
    static constexpr int TEAM = W * T;                           // 128 threads per team
    static constexpr int LPW = 32 / W;                           // threads of one column inside a warp
    static constexpr int BUF_BYTES = P::XPAD * W * 16;           // a tile buffer doubles as the exchange space
    static constexpr int NBUF = 3;
    static constexpr int THREADS = 2 * TEAM;
    static constexpr int TWB = round_up_c(P::TW_BYTES, 128);
    static constexpr size_t SMEM = PIPE_HEADER + TWB + (size_t)NBUF * BUF_BYTES;
    static_assert((TEAM / 32) * LPW == T, "team shape");
    static_assert(SMEM <= PIPE_SMEM_MAX, "tile ring does not fit");
};

// SQ: nx == ny == N (compile-time row stride).  YBE > 0: no column passes |ky| >= 2 T YBE (yband of ColArgs),
// known at compile time: the pair slots e in [YBE, 32 - YBE) are zero after the propagator.
template <int N, int MODE, bool SQ, int YBE>
__global__ void __launch_bounds__(ColPkCfg<N>::THREADS, 1) col_pk_kernel(ColArgs g)
{
    using C = ColPkCfg<N>;
    using P = typename C::P;
    constexpr int T = P::T, W = C::W;
    const int nx = SQ ? N : g.nx;
    constexpr bool LOADS = (MODE != COL_MS_INIT);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw);                    // [NBUF]
    float2* tab = reinterpret_cast<float2*>(smem_raw + PIPE_HEADER);
    unsigned char* bufs = smem_raw + PIPE_HEADER + C::TWB;
    const int tid = threadIdx.x, tm = tid / C::TEAM, tt = tid % C::TEAM;
    const int lane = tt & 31, c = lane % W, t = (tt >> 5) * C::LPW + lane / W;

    pk::fill_tables<P>(tab, g.tw_y, tid, C::THREADS);
    if (LOADS && tid == 0) {
        for (int b = 0; b < C::NBUF; ++b) mbar_init(&full[b], C::TEAM);
        mbar_fence_init();
    }
    __syncthreads();
    griddep_wait();                          // the previous kernel of the slice loop has completed (pipe_ptx.cuh)

    const int xb = g.xband;
    const int tiles_half = xb / W, tiles_per_wave = 2 * tiles_half;
    const long long n_items = (long long)g.n_waves * tiles_per_wave;
    const long long n_local = (n_items > blockIdx.x) ? (n_items - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    auto locate = [&](long long k, int& w, int& kx0) {
        const long long item = blockIdx.x + k * (long long)gridDim.x;
        w = (int)(item / tiles_per_wave);
        const int j = (int)(item % tiles_per_wave);
        kx0 = j < tiles_half ? j * W : nx - xb + (j - tiles_half) * W;
    };
    // all threads of a team: start the copies of local item k into buffer k % NBUF (rows in natural order)
    auto load = [&](long long k) {
        int w, kx0;
        locate(k, w, kx0);
        const float2* src = g.a + (size_t)w * N * nx + kx0;
        float2* buf = reinterpret_cast<float2*>(bufs + (size_t)(k % C::NBUF) * C::BUF_BYTES);
        constexpr int CH = W / 2;                                 // 16-byte chunks per row
#pragma unroll
        for (int i = 0; i < N * CH / C::TEAM; ++i) {
            const int q = tt + i * C::TEAM;
            const int row = q / CH, cc = q % CH;
            cp_async16(buf + row * W + 2 * cc, src + (size_t)row * nx + 2 * cc);
        }
        cp_async_arrive(&full[k % C::NBUF]);
    };
    if (LOADS) {
        if (tm == 0) { if (n_local > 0) load(0); if (n_local > 2) load(2); }
        else         { if (n_local > 1) load(1); }
    }
    auto sync = [&] { named_barrier(1 + tm, C::TEAM); };

    for (long long k = tm; k < n_local; k += 2) {
        int w, kx0;
        locate(k, w, kx0);
        const int kxi = kx0 + c;                                   // array slot of this thread's column
        const int bi = LOADS ? (int)(k % C::NBUF) : tm;
        unsigned char* buf = bufs + (size_t)bi * C::BUF_BYTES;
        const pk::Xchg16 sm{ reinterpret_cast<float4*>(buf) + c, W };
        C2 p[32];

        if (MODE == COL_MS_INIT) {
            // Psi0(kx, ky) = A_k exp(-i chi_k) exp(-2 pi i (kx xp / lx + ky yp / ly)) at ky = 2 j, 2 j + 1
            const int pr = g.probe0 + w;
            const int pxi = pr % g.probes_x, pyi = pr / g.probes_x;
            const float2 ex = __ldg(g.phase_x + (size_t)pxi * nx + kxi);
            const float4* ap = reinterpret_cast<const float4*>(g.aperture_t + (size_t)kxi * N);
            const float4* ey = reinterpret_cast<const float4*>(g.phase_y + (size_t)pyi * N);
#pragma unroll
            for (int e = 0; e < 32; ++e) {
                const int j = t + T * e;
                const float4 a = __ldg(ap + j), y = __ldg(ey + j);
                const float2 v0 = cmul(cmul(make_float2(a.x, a.y), ex), make_float2(y.x, y.y));
                const float2 v1 = cmul(cmul(make_float2(a.z, a.w), ex), make_float2(y.z, y.w));
                p[e] = { make_float2(v0.y, v1.y), make_float2(v0.x, v1.x) };       // (im, re): inverse = swapped forward
            }
        } else {
            float2 v[64];
            mbar_wait(&full[bi], (unsigned)((k / C::NBUF) & 1));
            const float2* tile = reinterpret_cast<const float2*>(buf) + c;
#pragma unroll
            for (int e = 0; e < 64; ++e) v[e] = tile[(t + T * e) * W];
            pk::fft_dif<P, 32>(v, p, tab, t, sm, sync);
            // Fresnel propagator with the 2/3 band-limit (Eq. 2; BASELINE.json) at ky = 2 j, 2 j + 1
            const float2 pxv = __ldg(g.prop_x + kxi);
            const int lim = __ldg(g.ky_lim + kxi);
            const float4* py4 = reinterpret_cast<const float4*>(g.prop_y);
#pragma unroll
            for (int e = 0; e < 32; ++e) {
                if (YBE > 0 && e >= YBE && e < 32 - YBE) { p[e] = { make_float2(0.f, 0.f), make_float2(0.f, 0.f) }; continue; }
                const int m0 = 2 * (t + T * e);
                const int ky0 = e < 16 ? m0 : N - m0, ky1 = e < 16 ? m0 + 1 : N - m0 - 1;     // |ky|
                const float4 q = __ldg(py4 + t + T * e);
                float2 pr0 = cmul(pxv, make_float2(q.x, q.y)), pr1 = cmul(pxv, make_float2(q.z, q.w));
                if (ky0 > lim) pr0 = make_float2(0.f, 0.f);
                if (ky1 > lim) pr1 = make_float2(0.f, 0.f);
                p[e] = pk::cmul2(p[e], make_float2(pr0.x, pr1.x), make_float2(pr0.y, pr1.y));
                if (MODE == COL_STEP) p[e] = pk::cswap(p[e]);
            }
        }

        if (MODE == COL_STEP || MODE == COL_MS_INIT) {
            float2 v[64];
            pk::fft_dit<P, 32>(p, v, tab, t, sm, sync);
            float2* dst = g.a + (size_t)w * N * nx + kxi;
            if (LOADS && k + C::NBUF < n_local) {
                // refill copies and tile stores interleaved (two stores, one 16-byte copy), so that neither kind
                // queues up alone in the LSU
                sync();                              // every thread of the team is past its last exchange read
                int w2, kx2;
                locate(k + C::NBUF, w2, kx2);
                const float2* src = g.a + (size_t)w2 * N * nx + kx2;
                float2* nbuf = reinterpret_cast<float2*>(bufs + (size_t)((k + C::NBUF) % C::NBUF) * C::BUF_BYTES);
                constexpr int CH = W / 2;
                static_assert(N * CH / C::TEAM == 32, "interleave ratio");
#pragma unroll
                for (int i = 0; i < 32; ++i) {
                    dst[(size_t)(t + T * (2 * i)) * nx] = make_float2(v[2 * i].y, v[2 * i].x);
                    dst[(size_t)(t + T * (2 * i + 1)) * nx] = make_float2(v[2 * i + 1].y, v[2 * i + 1].x);
                    const int q = tt + i * C::TEAM;
                    const int row = q / CH, cc = q % CH;
                    cp_async16(nbuf + row * W + 2 * cc, src + (size_t)row * nx + 2 * cc);
                }
                cp_async_arrive(&full[(k + C::NBUF) % C::NBUF]);
            } else {
#pragma unroll
                for (int e = 0; e < 64; ++e) dst[(size_t)(t + T * e) * nx] = make_float2(v[e].y, v[e].x);
            }
        } else {
            if (k + C::NBUF < n_local) {
                sync();
                load(k + C::NBUF);
            }
            // detector-plane intensity, ky contiguous
            float2* dst = reinterpret_cast<float2*>(g.intensity + ((size_t)w * nx + kxi) * N);
#pragma unroll
            for (int e = 0; e < 32; ++e) {
                const float2 i2 = pk::fma2(p[e].x, p[e].x, pk::mul2(p[e].y, p[e].y));
                dst[t + T * e] = make_float2(i2.x * g.scale, i2.y * g.scale);
            }
        }
    }
}

// =============================================================================
// Column pass on the blocked layout "B8" (top of this file)
// =============================================================================
// A CTA of 8 warps works on one tile [N rows] x [8 columns] = 128 KB, which is one contiguous run of the blocked
// layout: a few bulk copies (TMA engine, mbarrier transaction count) land it in shared memory, every thread takes
// its 64 points into registers, and the landing buffer is refilled with the next tile at once, so the fetch of
// tile k + 1 overlaps the computation of tile k.  The half-length transforms exchange through a separate 8-byte
// plane used twice (real parts, then imaginary parts).  The y-factor of the propagator sits in shared memory (with
// 216 KB of it in use there is next to no L1 left).
// One team of 256 threads owns all 8 columns, so a warp's store instruction covers 4 rows x 64 B = 256 contiguous
// bytes.  (Two teams of 128 threads on columns 0-3 / 4-7 of the same tile, skewed by half a tile so that one
// team's butterflies overlap the other's exchanges, measured slower: 14.6 ms against 13.9 ms per launch -- their
// stores are 32-byte row segments again and their landing reads conflict two-way.)

template <int N>
struct ColB8Cfg {
    using P = pk::PkPlan<N>;
    static constexpr int T = P::T;                               // threads per column
    static constexpr int W = 8;                                  // columns per tile
    static constexpr int THREADS = W * T;
    static constexpr int TILE_BYTES = N * W * 8;
    static constexpr int X_BYTES = P::XPAD * W * 8;              // 8-byte exchange planes of all columns, used in two phases
    static constexpr int TWB = round_up_c(P::TW_BYTES, 128);
    static constexpr int PYB = N * 8;
    static constexpr size_t SMEM = PIPE_HEADER + TWB + PYB + (size_t)TILE_BYTES + X_BYTES;
    static constexpr int CHUNKS = 4;                             // bulk copies per tile
    static_assert(THREADS == 256, "team shape");
    static_assert(SMEM <= PIPE_SMEM_MAX, "tile + exchange planes do not fit");
};

template <int N, int MODE, int YBE>
__global__ void __launch_bounds__(ColB8Cfg<N>::THREADS, 1) col_b8_kernel(ColArgs g)
{
    using C = ColB8Cfg<N>;
    using P = typename C::P;
    constexpr int T = P::T, W = C::W;
    constexpr int LPW = 32 / W;                                   // threads of one column inside a warp
    static_assert((C::THREADS / 32) * LPW == T, "team shape");
    constexpr bool LOADS = (MODE != COL_MS_INIT);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw);
    float2* tab = reinterpret_cast<float2*>(smem_raw + PIPE_HEADER);
    float4* py_s = reinterpret_cast<float4*>(smem_raw + PIPE_HEADER + C::TWB);            // pairs (P_y[2j], P_y[2j+1])
    float2* tile = reinterpret_cast<float2*>(smem_raw + PIPE_HEADER + C::TWB + C::PYB);    // [N][8]
    float2* xch = reinterpret_cast<float2*>(smem_raw + PIPE_HEADER + C::TWB + C::PYB + C::TILE_BYTES);
    const int tid = threadIdx.x, lane = tid & 31;
    const int c = lane % W, t = (tid >> 5) * LPW + lane / W;

    pk::fill_tables<P>(tab, g.tw_y, tid, C::THREADS);
    if (MODE != COL_MS_INIT)
        for (int i = tid; i < N; i += C::THREADS) reinterpret_cast<float2*>(py_s)[i] = __ldg(g.prop_y + i);
    if (LOADS && tid == 0) { mbar_init(full, 1); mbar_fence_init(); }
    __syncthreads();
    griddep_wait();                          // the previous kernel of the slice loop has completed (pipe_ptx.cuh)

    const int xb = g.xband, nx = g.nx;
    const int tiles_per_wave = 2 * xb / W;
    const size_t wave_stride = (size_t)N * nx;
    const long long n_items = (long long)g.n_waves * tiles_per_wave;
    const long long n_local = (n_items > blockIdx.x) ? (n_items - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    auto locate = [&](long long k, int& w, int& j) {
        const long long item = blockIdx.x + k * (long long)gridDim.x;
        w = (int)(item / tiles_per_wave);
        j = (int)(item % tiles_per_wave);
    };
    // one thread: start the bulk copies of local item k into the landing buffer
    auto load = [&](long long k) {
        int w, j;
        locate(k, w, j);
        const unsigned char* src = reinterpret_cast<const unsigned char*>(g.a + (size_t)w * wave_stride + (size_t)j * N * W);
        mbar_expect_tx(full, (unsigned)C::TILE_BYTES);
#pragma unroll
        for (int i = 0; i < C::CHUNKS; ++i)
            bulk_g2s(reinterpret_cast<unsigned char*>(tile) + i * (C::TILE_BYTES / C::CHUNKS),
                     src + i * (C::TILE_BYTES / C::CHUNKS), (unsigned)(C::TILE_BYTES / C::CHUNKS), full);
    };
    if (LOADS && tid == 0 && n_local > 0) load(0);
    auto sync = [] { __syncthreads(); };
    const pk::XchgPhase sm{ xch + c, W };

    for (long long k = 0; k < n_local; ++k) {
        int w, j;
        locate(k, w, j);
        const int jc = j * W + c;                                  // compact column
        const int kxi = jc < xb ? jc : nx - 2 * xb + jc;           // its array slot along kx
        C2 p[32];

        if (MODE == COL_MS_INIT) {
            // Psi0(kx, ky) = A_k exp(-i chi_k) exp(-2 pi i (kx xp / lx + ky yp / ly)) at ky = 2 j, 2 j + 1
            const int pr = g.probe0 + w;
            const int pxi = pr % g.probes_x, pyi = pr / g.probes_x;
            const float2 ex = __ldg(g.phase_x + (size_t)pxi * nx + kxi);
            const float4* ap = reinterpret_cast<const float4*>(g.aperture_t + (size_t)kxi * N);
            const float4* ey = reinterpret_cast<const float4*>(g.phase_y + (size_t)pyi * N);
#pragma unroll
            for (int e = 0; e < 32; ++e) {
                const int m = t + T * e;
                const float4 a = __ldg(ap + m), y = __ldg(ey + m);
                const float2 v0 = cmul(cmul(make_float2(a.x, a.y), ex), make_float2(y.x, y.y));
                const float2 v1 = cmul(cmul(make_float2(a.z, a.w), ex), make_float2(y.z, y.w));
                p[e] = { make_float2(v0.y, v1.y), make_float2(v0.x, v1.x) };       // (im, re): inverse = swapped forward
            }
        } else {
            float2 v[64];
            // per-column propagator factor and band limit: requested now, used between the transforms
            const float2 pxv = __ldg(g.prop_x + kxi);
            const int lim = __ldg(g.ky_lim + kxi);
            mbar_wait(full, (unsigned)(k & 1));
#pragma unroll
            for (int e = 0; e < 64; ++e) v[e] = tile[(t + T * e) * W + c];
            // the landing buffer is free once every thread has taken its points: refill it with the next tile
            sync();
            if (tid == 0 && k + 1 < n_local) { fence_proxy_async(); load(k + 1); }
            pk::dif_pre<P, 32>(v, p, tab, t);
            pk::fft_half<P, false>(p, tab, t, sm, sync);        // the barrier after the landing reads covers the exchange plane
            // Fresnel propagator with the 2/3 band-limit (Eq. 2; BASELINE.json) at ky = 2 j, 2 j + 1
#pragma unroll
            for (int e = 0; e < 32; ++e) {
                if (YBE > 0 && e >= YBE && e < 32 - YBE) { p[e] = { make_float2(0.f, 0.f), make_float2(0.f, 0.f) }; continue; }
                const int m0 = 2 * (t + T * e);
                const int ky0 = e < 16 ? m0 : N - m0, ky1 = e < 16 ? m0 + 1 : N - m0 - 1;     // |ky|
                const float4 q = py_s[t + T * e];
                float2 pr0 = cmul(pxv, make_float2(q.x, q.y)), pr1 = cmul(pxv, make_float2(q.z, q.w));
                if (ky0 > lim) pr0 = make_float2(0.f, 0.f);
                if (ky1 > lim) pr1 = make_float2(0.f, 0.f);
                p[e] = pk::cmul2(p[e], make_float2(pr0.x, pr1.x), make_float2(pr0.y, pr1.y));
                if (MODE == COL_STEP) p[e] = pk::cswap(p[e]);
            }
        }

        if (MODE == COL_STEP || MODE == COL_MS_INIT) {
            float2 v[64];
            pk::fft_half<P>(p, tab, t, sm, sync);
            pk::dit_post<P, 32>(p, v, tab, t);
            float2* dst = g.a + (size_t)w * wave_stride + (size_t)j * N * W + c;
#pragma unroll
            for (int e = 0; e < 64; ++e) dst[(t + T * e) * W] = make_float2(v[e].y, v[e].x);
        } else {
            // detector-plane intensity, ky contiguous
            float2* dst = reinterpret_cast<float2*>(g.intensity + ((size_t)w * nx + kxi) * N);
#pragma unroll
            for (int e = 0; e < 32; ++e) {
                const float2 i2 = pk::fma2(p[e].x, p[e].x, pk::mul2(p[e].y, p[e].y));
                dst[t + T * e] = make_float2(i2.x * g.scale, i2.y * g.scale);
            }
        }
    }
}

template <int N, int MODE, int YBE>
static cudaError_t launch_col_b8_s(const ColArgs& g, cudaStream_t stream)
{
    using C = ColB8Cfg<N>;
    auto kern = col_b8_kernel<N, MODE, YBE>;
    static PerDevice once{};
    if (cudaError_t e = opt_in_smem(kern, C::SMEM, once); e != cudaSuccess) return e;
    if (g.xband % C::W) return cudaErrorInvalidValue;
    const long long n_items = (long long)g.n_waves * (2 * g.xband / C::W);
    if (n_items == 0) return cudaSuccess;
    long long grid = n_items;
    if (grid > num_sms()) grid = num_sms();
    return launch_pdl(kern, (unsigned)grid, C::THREADS, C::SMEM, stream, g);
}

template <int N, int MODE>
static cudaError_t launch_col_b8_t(const ColArgs& g, cudaStream_t stream)
{
    constexpr int YB = DefaultBand<N>::XB, T = N / 64;
    if (g.yband == YB) return launch_col_b8_s<N, MODE, YB / (2 * T)>(g, stream);
    return launch_col_b8_s<N, MODE, 0>(g, stream);
}

static cudaError_t launch_col_b8(ColMode mode, const ColArgs& g, cudaStream_t stream)
{
    if (g.ny != 2048) return cudaErrorInvalidValue;
    switch (mode) {
        case COL_STEP:     return launch_col_b8_t<2048, COL_STEP>(g, stream);
        case COL_MS_INIT:  return launch_col_b8_t<2048, COL_MS_INIT>(g, stream);
        case COL_MS_FINAL: return launch_col_b8_t<2048, COL_MS_FINAL>(g, stream);
        default: break;
    }
    return cudaErrorInvalidValue;
}

template <int N, int MODE, bool SQ, int YBE>
static cudaError_t launch_col_pk_s(const ColArgs& g, cudaStream_t stream)
{
    using C = ColPkCfg<N>;
    auto kern = col_pk_kernel<N, MODE, SQ, YBE>;
    static PerDevice once{};
    if (cudaError_t e = opt_in_smem(kern, C::SMEM, once); e != cudaSuccess) return e;
    if (g.xband % C::W || g.nx % C::W) return cudaErrorInvalidValue;
    const long long n_items = (long long)g.n_waves * (2 * g.xband / C::W);
    if (n_items == 0) return cudaSuccess;
    long long grid = (n_items + 1) / 2;                             // at least one tile per team
    if (grid > num_sms()) grid = num_sms();
    return launch_pdl(kern, (unsigned)grid, C::THREADS, C::SMEM, stream, g);
}

template <int N, int MODE>
static cudaError_t launch_col_pk_t(const ColArgs& g, cudaStream_t stream)
{
    constexpr int YB = DefaultBand<N>::XB, T = N / 64;
    static_assert(YB % (2 * T) == 0, "default band must be a whole number of pair slots");
    if (g.nx == N && g.yband == YB) return launch_col_pk_s<N, MODE, true, YB / (2 * T)>(g, stream);
    if (g.nx == N) return launch_col_pk_s<N, MODE, true, 0>(g, stream);
    return launch_col_pk_s<N, MODE, false, 0>(g, stream);
}

template <int N>
static cudaError_t launch_col_pk_n(ColMode mode, const ColArgs& g, cudaStream_t stream)
{
    switch (mode) {
        case COL_STEP:     return launch_col_pk_t<N, COL_STEP>(g, stream);
        case COL_MS_INIT:  return launch_col_pk_t<N, COL_MS_INIT>(g, stream);
        case COL_MS_FINAL: return launch_col_pk_t<N, COL_MS_FINAL>(g, stream);
        default: break;
    }
    return cudaErrorInvalidValue;
}

cudaError_t launch_col_pk(ColMode mode, const ColArgs& g, cudaStream_t stream)
{
    if (g.xband < 4 || 2 * g.xband > g.nx) return cudaErrorInvalidValue;
    if (g.blocked) return launch_col_b8(mode, g, stream);
    switch (g.ny) {
        case 1024: return launch_col_pk_n<1024>(mode, g, stream);
        case 2048: return launch_col_pk_n<2048>(mode, g, stream);
    }
    return cudaErrorInvalidValue;
}

}  // namespace prism
