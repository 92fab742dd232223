// slice_pipe_col.cu -- software-pipelined column pass of the slice step (columns of 256 .. 1024 points).
//
// PAPER.md:80 Eq. (2)  Psi <- Psi * exp(-i pi lambda q^2 t)  (propagation), "done in Fourier space"
//
// Column pass FFT_y . P . IFFT_y on mixed space A[w][y][kx] (see slice_pass.cu for the two-pass structure):
//
//  * every thread holds E = 32 points, so columns up to 1024 points need ONE shared-memory exchange
//    per transform, and inter-stage twiddles come from a transposed shared table;
//  * two teams of 256 threads per CTA alternate over [N rows] x [W columns] tiles of 8192 points held
//    in a three-buffer ring filled by 16-byte cp.async copies that signal an mbarrier; a lane owns one
//    column of the tile and consecutive lanes consecutive columns, so every shared-memory access of
//    the transforms is a contiguous run and results are stored from registers as 64-byte (W = 8)
//    row segments;
//  * band-limit: after the column pass everything with |kx| > kx_max is exactly zero (2/3 rule,
//    BASELINE.json), so the pass runs on the 2 xband / W in-band tiles of a wave only.
//
// 2048-point columns run on the packed kernels of slice_pk.cu.
#include "fft_core.cuh"
#include "pipe_plan.cuh"
#include "prism_internal.h"
#include "pipe_ptx.cuh"

namespace prism {

constexpr int COL_TILE_PTS = 8192;

// =============================================================================
// Column pass
// =============================================================================
template <class P>
struct ColCfg {
    static constexpr int TILE_PTS = COL_TILE_PTS;
    static constexpr int W = TILE_PTS / P::N;                    // columns per tile: 32, 16, 8, 4
    static constexpr int TEAM = TILE_PTS / P::E;                 // 256 threads per team
    static constexpr int LPW = 32 / W;                           // threads of one column inside a warp
    static constexpr int ROWS = P::N + P::N / P::R1;             // padded rows
    static constexpr int BUF = ROWS * W;                         // float2 per buffer
    static constexpr int NT = 512 / TEAM;                        // teams per CTA
    static constexpr int THREADS = NT * TEAM;
    static constexpr int NBUF_FIT = (PIPE_SMEM_MAX - PIPE_HEADER - round_up_c(SmemTwiddles<P>::COUNT * 8, 128)) / (BUF * 8);
    static constexpr int NBUF = NBUF_FIT < NT + NT / 2 ? NBUF_FIT : NT + NT / 2;   // 3 buffers for 2 teams, 6 for 4
    static constexpr int TWB = round_up_c(SmemTwiddles<P>::COUNT * 8, 128);
    // the y-factor of the propagator sits in shared memory when it fits beside the tile ring (keeps 22 loads per
    // thread and tile out of the LSU's global-memory queue)
    static constexpr bool PY_SMEM = PIPE_HEADER + TWB + (size_t)NBUF * BUF * 8 + P::N * 8 <= PIPE_SMEM_MAX;
    static constexpr int PYB = PY_SMEM ? P::N * 8 : 0;
    static constexpr size_t SMEM = PIPE_HEADER + TWB + PYB + (size_t)NBUF * BUF * 8;
    static_assert(TEAM / 32 * LPW == P::T, "team shape");
    static_assert(SMEM <= PIPE_SMEM_MAX, "tile ring does not fit");
};

// column c of a tile buffer: element idx at base[(idx + idx / R1) * W]   (base already offset by c)
template <class P, int W, int TEAM>
struct ColSm {
    float2* base;
    int bar_id;
    __device__ __forceinline__ static int phys(int idx) { return idx + idx / P::R1; }
    __device__ __forceinline__ void  st(int idx, float2 v) const { base[phys(idx) * W] = v; }
    __device__ __forceinline__ void  st2(int idx, float2 v0, float2 v1) const { st(idx, v0); st(idx + 1, v1); }
    __device__ __forceinline__ float2 ld(int idx) const { return base[phys(idx) * W]; }
    __device__ __forceinline__ void sync() const { named_barrier(bar_id, TEAM); }
};

// SQ: nx == ny == N, so every row stride is a compile-time constant (immediate offsets, no 64-bit index math).
// YBE > 0: no column passes |ky| >= YBE * T (yband of ColArgs), known at compile time.
template <class P, int MODE, bool SQ, int YBE>
__global__ void __launch_bounds__(ColCfg<P>::THREADS, 1) col_pipe_kernel(ColArgs g)
{
    using C = ColCfg<P>;
    constexpr int E = P::E, T = P::T, N = P::N, W = C::W;
    const int nx = SQ ? N : g.nx;
    constexpr bool LOADS = (MODE != COL_MS_INIT);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw);                    // [NBUF]
    float2* twtab = reinterpret_cast<float2*>(smem_raw + PIPE_HEADER);
    float2* py_s = reinterpret_cast<float2*>(smem_raw + PIPE_HEADER + C::TWB);
    float2* bufs = reinterpret_cast<float2*>(smem_raw + PIPE_HEADER + C::TWB + C::PYB);
    const int tid = threadIdx.x, tm = tid / C::TEAM, tt = tid % C::TEAM;
    const int lane = tt & 31, c = lane % W, t = (tt >> 5) * C::LPW + lane / W;

    SmemTwiddles<P>::fill(twtab, g.tw_y, tid, C::THREADS);
    if (C::PY_SMEM && MODE != COL_MS_INIT)
        for (int i = tid; i < N; i += C::THREADS) py_s[i] = __ldg(g.prop_y + i);
    if (LOADS && tid == 0) {
        for (int b = 0; b < C::NBUF; ++b) mbar_init(&full[b], C::TEAM);
        mbar_fence_init();
    }
    __syncthreads();
    SmemTwiddles<P> tw;
    tw.bind(twtab, t);
    griddep_wait();                          // the previous kernel of the slice loop has completed (pipe_ptx.cuh)

    const int xb = g.xband;
    const int tiles_half = xb / W, tiles_per_wave = 2 * tiles_half;
    const long long n_items = (long long)g.n_waves * tiles_per_wave;
    // local item k of this CTA is global item blockIdx.x + k * gridDim.x
    const long long n_local = (n_items > blockIdx.x) ? (n_items - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    auto locate = [&](long long k, int& w, int& kx0) {
        const long long item = blockIdx.x + k * (long long)gridDim.x;
        w = (int)(item / tiles_per_wave);
        const int j = (int)(item % tiles_per_wave);
        kx0 = j < tiles_half ? j * W : nx - xb + (j - tiles_half) * W;
    };
    // all threads of a team: start the copies of local item k into buffer k % NBUF
    auto load = [&](long long k) {
        int w, kx0;
        locate(k, w, kx0);
        const float2* src = g.a + (size_t)w * N * nx + kx0;
        float2* buf = bufs + (size_t)(k % C::NBUF) * C::BUF;
        // 16-byte chunk q = tt + i TEAM of the tile: row q / CH, chunk q % CH of the row.  TEAM / CH rows per step, a
        // multiple of R1, so both addresses advance by constants (no per-copy index arithmetic)
        constexpr int CH = W / 2, STEP = C::TEAM / CH;
        static_assert(C::TEAM % CH == 0 && STEP % P::R1 == 0, "copy pattern");
        const int r0 = tt / CH, cc = tt % CH;
        const float2* s0 = src + (size_t)r0 * nx + 2 * cc;
        float2* d0 = buf + (r0 + r0 / P::R1) * W + 2 * cc;
#pragma unroll
        for (int i = 0; i < N / STEP; ++i)
            cp_async16(d0 + i * (STEP + STEP / P::R1) * W, s0 + (size_t)i * STEP * nx);
        cp_async_arrive(&full[k % C::NBUF]);
    };
    if (LOADS) {
#pragma unroll
        for (int i = 0; i < C::NBUF; ++i)
            if (i % C::NT == tm && i < n_local) load(i);
    }

    for (long long k = tm; k < n_local; k += C::NT) {
        int w, kx0;
        locate(k, w, kx0);
        const int kxi = kx0 + c;                                   // array slot of this thread's column
        const int bi = LOADS ? (int)(k % C::NBUF) : tm;
        const ColSm<P, W, C::TEAM> sm{ bufs + (size_t)bi * C::BUF + c, 1 + tm };
        float2 v[E];

        if (MODE == COL_MS_INIT) {
            // Psi0(kx, ky) = A_k exp(-i chi_k) exp(-2 pi i (kx xp / lx + ky yp / ly))
            const int p = g.probe0 + w;
            const int pxi = p % g.probes_x, pyi = p / g.probes_x;
            const float2 ex = __ldg(g.phase_x + (size_t)pxi * nx + kxi);
            const float2* ap = g.aperture_t + (size_t)kxi * N;
            const float2* ey = g.phase_y + (size_t)pyi * N;
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const int m = t + T * e;
                v[e] = cmul(cmul(__ldg(ap + m), ex), __ldg(ey + m));
            }
        } else {
            mbar_wait(&full[bi], (unsigned)((k / C::NBUF) & 1));
#pragma unroll
            for (int e = 0; e < E; ++e) v[e] = sm.ld(t + T * e);
            fft_forward<P>(v, tw, t, sm);
            // Fresnel propagator with the 2/3 band-limit (Eq. 2; BASELINE.json).  With YBE > 0 the
            // register slots e in [YBE, E - YBE) hold |ky| beyond every column's limit: zero without any work.
            const float2 pxv = __ldg(g.prop_x + kxi);
            const int lim = __ldg(g.ky_lim + kxi);
#pragma unroll
            for (int e = 0; e < E; ++e) {
                if (YBE > 0 && e >= YBE && e < E - YBE) { v[e] = make_float2(0.f, 0.f); continue; }
                const int m = t + T * e;
                const int ky = e < E / 2 ? m : N - m;           // |ky|
                const float2 pr = cmul(pxv, C::PY_SMEM ? py_s[m] : __ldg(g.prop_y + m));
                v[e] = (ky <= lim) ? cmul(v[e], pr) : make_float2(0.f, 0.f);
            }
        }
        if (MODE == COL_STEP || MODE == COL_MS_INIT) fft_inverse<P>(v, tw, t, sm);

        // Order of the tile's stores and of the refill of its buffer: with 64-byte row segments (1024-point columns)
        // the stores go first, so that they do not queue behind the cp.async copies in the LSU (1.49 -> 1.35 ms); with
        // wider segments the earlier prefetch wins (512 points: 0.39 ms against 0.42 ms)
        constexpr bool STORE_FIRST = (N >= 1024);
        auto refill = [&] {
            if (LOADS && k + C::NBUF < n_local) {
                sm.sync();                           // every thread of the team is past its last exchange read
                load(k + C::NBUF);
            }
        };
        if (!STORE_FIRST) refill();
        if (MODE == COL_STEP || MODE == COL_MS_INIT) {
            float2* dst = g.a + (size_t)w * N * nx + kxi;
#pragma unroll
            for (int e = 0; e < E; ++e) dst[(size_t)(t + T * e) * nx] = v[e];
            if (STORE_FIRST) refill();
        } else {
            if (STORE_FIRST) refill();
            // detector-plane intensity, ky contiguous
            float* dst = g.intensity + ((size_t)w * nx + kxi) * N;
#pragma unroll
            for (int e = 0; e < E; ++e)
                dst[t + T * e] = (v[e].x * v[e].x + v[e].y * v[e].y) * g.scale;
        }
    }
}

template <class P, int MODE, bool SQ, int YBE>
static cudaError_t launch_col_pipe_s(const ColArgs& g, cudaStream_t stream)
{
    using C = ColCfg<P>;
    auto kern = col_pipe_kernel<P, MODE, SQ, YBE>;
    static PerDevice once{};
    if (cudaError_t e = opt_in_smem(kern, C::SMEM, once); e != cudaSuccess) return e;
    if (g.xband % C::W || g.nx % C::W) return cudaErrorInvalidValue;
    const long long n_items = (long long)g.n_waves * (2 * g.xband / C::W);
    if (n_items == 0) return cudaSuccess;
    long long grid = (n_items + C::NT - 1) / C::NT;                 // at least one tile per team
    if (grid > num_sms()) grid = num_sms();
    return launch_pdl(kern, (unsigned)grid, C::THREADS, C::SMEM, stream, g);
}

template <class P, int MODE>
static cudaError_t launch_col_pipe_t(const ColArgs& g, cudaStream_t stream)
{
    constexpr int YB = DefaultBand<P::N>::XB;
    if (g.nx == P::N && g.yband == YB) return launch_col_pipe_s<P, MODE, true, YB / P::T>(g, stream);
    if (g.nx == P::N) return launch_col_pipe_s<P, MODE, true, 0>(g, stream);
    return launch_col_pipe_s<P, MODE, false, 0>(g, stream);
}

template <int N>
static cudaError_t launch_col_pipe_n(ColMode mode, const ColArgs& g, cudaStream_t stream)
{
    using P = typename PipePlan<N>::type;
    switch (mode) {
        case COL_STEP:     return launch_col_pipe_t<P, COL_STEP>(g, stream);
        case COL_MS_INIT:  return launch_col_pipe_t<P, COL_MS_INIT>(g, stream);
        case COL_MS_FINAL: return launch_col_pipe_t<P, COL_MS_FINAL>(g, stream);
        default: break;
    }
    return cudaErrorInvalidValue;
}

cudaError_t launch_col_pipe(ColMode mode, const ColArgs& g, cudaStream_t stream)
{
    if (g.xband < 4 || 2 * g.xband > g.nx) return cudaErrorInvalidValue;
    switch (g.ny) {
        case 256:  return launch_col_pipe_n<256>(mode, g, stream);
        case 512:  return launch_col_pipe_n<512>(mode, g, stream);
        case 1024: return launch_col_pipe_n<1024>(mode, g, stream);
    }
    return cudaErrorInvalidValue;
}

}  // namespace prism
