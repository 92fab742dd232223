// ms_resident.cu -- plain multislice with one probe per SM, resident from the probe spectrum to the ring sums
// ("resident multislice for N <= 512"; comparison path M1).
//
// PAPER.md:132 "The initial probe is translated to the probe position of interest, and then is alternately
//   transmitted and propagated through the sample ... alternating forward and inverse Fourier transforms with an
//   element-wise complex multiplication in between" ; PAPER.md:82 annular ring detectors.
//
// The per-pass kernels (slice_pipe_*.cu) run every slice of a probe batch as two launches; at 256^2 a launch
// lasts 15-20 us and is mostly prologue, first-load latency and tail.  Here ONE launch carries all probes through
// all slices: a CTA (one per SM) owns a probe -- its wave lives in a private [N][N] slot of the workspace that stays
// in L2 -- and alternates the same two passes on it,
//
//   row pass    : IFFT_x . t_s . FFT_x  on its N rows    (lines straight into registers, next lines prefetched)
//   column pass : FFT_y  . P   . IFFT_y on its 2 xb in-band columns (tiles [N][W] through shared memory, two teams)
//
// separated by __syncthreads only; it starts from the probe spectrum (no read), ends in |Psi|^2 (no inverse
// transform) and sums the rings itself.  Same arithmetic, tables and band-limit bookkeeping as the per-pass path
// (DESIGN.md section 6 scale bookkeeping); transmission functions of all slices are computed beforehand.
// (scalar complex adds: packed FADD2 butterflies measured slower here, 18.75 against 18.08 ms per 1024 probes of MS2)
#include "fft_core.cuh"
#include "pipe_ptx.cuh"
#include "prism_internal.h"

namespace prism {

template <int N>
struct MsCfg {
    using P = typename PlanFor<N>::type;                        // E = 16 points per thread
    static constexpr int E = P::E, T = P::T;
    static constexpr int THREADS = 512;
    static constexpr int LINES = THREADS / T;                    // rows per sweep of the row pass
    static constexpr int TEAM = 256, NTEAMS = THREADS / TEAM;
    static constexpr int W = TEAM / T;                           // columns per tile: 16 (N = 256), 8 (N = 512)
    static constexpr int ROWS = P::PADDED;
    static constexpr int BUF = ROWS * W;                         // float2 per tile buffer
    static constexpr int TWN = SmemTwiddles<P>::COUNT;
    static constexpr size_t XCH_BYTES = (size_t)LINES * P::PADDED * 8;            // row-pass exchange space
    static constexpr size_t TILE_BYTES = (size_t)NTEAMS * 2 * BUF * 8;            // two buffers per team
    static constexpr size_t WORK_BYTES = XCH_BYTES > TILE_BYTES ? XCH_BYTES : TILE_BYTES;   // the passes alternate
    static constexpr size_t SMEM = (size_t)TWN * 8 + (size_t)N * 8 + WORK_BYTES;
    static_assert(N % LINES == 0 && T <= 32 && W >= 2, "shape");
    static_assert(SMEM <= 227 * 1024, "does not fit");
};

// column c of a tile buffer: element idx at base[pad16(idx) * W] (base already offset by c); a column's threads sit
// in different warps, so its exchanges are fenced by the team's named barrier
template <int W, int TEAM>
struct ColLine {
    float2* base;
    int bar_id;
    __device__ __forceinline__ void  st(int idx, float2 v) const { base[pad16(idx) * W] = v; }
    __device__ __forceinline__ void  st2(int idx, float2 v0, float2 v1) const { st(idx, v0); st(idx + 1, v1); }
    __device__ __forceinline__ float2 ld(int idx) const { return base[pad16(idx) * W]; }
    __device__ __forceinline__ void sync() const { named_barrier(bar_id, TEAM); }
};

__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int PENDING> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(PENDING) : "memory"); }

// XBE / YBE > 0: xband = XBE * T and yband = YBE * T are known at compile time (register slots beyond the band are
// constants); 0: tested per element.
template <int N, int XBE, int YBE>
__global__ void __launch_bounds__(MsCfg<N>::THREADS, 1) ms_resident_kernel(MsResidentArgs g)
{
    using C = MsCfg<N>;
    using P = typename C::P;
    constexpr int E = C::E, T = C::T, W = C::W;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* twtab = reinterpret_cast<float2*>(smem_raw);
    float2* py_s = twtab + C::TWN;                                               // y-factor of the propagator
    float2* work = py_s + N;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    SmemTwiddles<P>::fill(twtab, g.tw, tid, C::THREADS);
    for (int i = tid; i < N; i += C::THREADS) py_s[i] = __ldg(g.prop_y + i);
    __syncthreads();

    const int xb = XBE > 0 ? XBE * T : g.xband;
    // ---- row pass roles ----
    const int rl = tid / T, rt = tid % T;                                        // line of the sweep, thread of the line
    SmemTwiddles<P> twr;
    twr.bind(twtab, rt);
    const LineSmem<P> rsm{ work + rl * P::PADDED, 1 };
    auto x_in_band = [&](int e) { return XBE > 0 ? (e < XBE || e >= E - XBE) : (rt + T * e < xb || rt + T * e >= N - xb); };
    // ---- column pass roles ----
    const int tm = tid / C::TEAM, tt = tid % C::TEAM;
    const int cc = tt % W, ct = tt / W;                                          // column of the tile, thread of the column
    SmemTwiddles<P> twc;
    twc.bind(twtab, ct);
    float2* my_bufs = work + (size_t)tm * 2 * C::BUF;
    const int tiles_half = xb / W, tiles = 2 * tiles_half;                       // in-band tiles of a wave
    const int my_tiles = tiles > tm ? (tiles - tm + C::NTEAMS - 1) / C::NTEAMS : 0;
    auto tile_kx0 = [&](int k) { const int j = tm + k * C::NTEAMS; return j < tiles_half ? j * W : N - xb + (j - tiles_half) * W; };

    float2* psi = g.psi + (size_t)blockIdx.x * N * N;                            // this CTA's wave slot
    float* inten = g.intensity + (size_t)blockIdx.x * N * N;

    // all threads of a team: start the copies of its local tile k into buffer k & 1
    auto load_tile = [&](int k) {
        const float2* src = psi + tile_kx0(k);
        float2* buf = my_bufs + (size_t)(k & 1) * C::BUF;
        constexpr int CH = W / 2;                                                // 16-byte chunks per row
#pragma unroll
        for (int i = 0; i < N * CH / C::TEAM; ++i) {
            const int q = tt + i * C::TEAM;
            const int row = q / CH, c2 = q % CH;
            cp_async16(buf + pad16(row) * W + 2 * c2, src + (size_t)row * N + 2 * c2);
        }
        cp_async_commit();
    };

    // mode 0: spectrum -> IFFT_y (no read); 1: FFT_y . P . IFFT_y; 2: FFT_y . P -> |.|^2 (no inverse)
    auto column_pass = [&](int mode, int probe) {
        if (mode != 0 && my_tiles > 0) load_tile(0);
        for (int k = 0; k < my_tiles; ++k) {
            const int kx0 = tile_kx0(k), kxi = kx0 + cc;
            const ColLine<W, C::TEAM> sm{ my_bufs + (size_t)(k & 1) * C::BUF + cc, 1 + tm };
            float2 v[E];
            if (mode == 0) {
                // Psi0(kx, ky) = A_k exp(-i chi_k) exp(-2 pi i (kx xp / lx + ky yp / ly))
                const int pxi = probe % g.probes_x, pyi = probe / g.probes_x;
                const float2 ex = __ldg(g.phase_x + (size_t)pxi * N + kxi);
                const float2* ap = g.aperture_t + (size_t)kxi * N;
                const float2* ey = g.phase_y + (size_t)pyi * N;
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    const int m = ct + T * e;
                    v[e] = cmul(cmul(__ldg(ap + m), ex), __ldg(ey + m));
                }
            } else {
                if (k + 1 < my_tiles) { load_tile(k + 1); cp_async_wait<1>(); } else { cp_async_wait<0>(); }
                sm.sync();                                   // every thread's copies of tile k have landed
#pragma unroll
                for (int e = 0; e < E; ++e) v[e] = sm.ld(ct + T * e);
                fft_forward<P>(v, twc, ct, sm);
                // Fresnel propagator with the 2/3 band-limit (Eq. 2; BASELINE.json)
                const float2 pxv = __ldg(g.prop_x + kxi);
                const int lim = __ldg(g.ky_lim + kxi);
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    if (YBE > 0 && e >= YBE && e < E - YBE) { v[e] = make_float2(0.f, 0.f); continue; }
                    const int m = ct + T * e;
                    const int ky = e < E / 2 ? m : N - m;    // |ky|
                    const float2 pr = cmul(pxv, py_s[m]);
                    v[e] = (ky <= lim) ? cmul(v[e], pr) : make_float2(0.f, 0.f);
                }
            }
            if (mode != 2) {
                fft_inverse<P>(v, twc, ct, sm);
                float2* dst = psi + kxi;
#pragma unroll
                for (int e = 0; e < E; ++e) dst[(size_t)(ct + T * e) * N] = v[e];
            } else {
                // detector-plane intensity, ky contiguous
                float* dst = inten + (size_t)kxi * N;
#pragma unroll
                for (int e = 0; e < E; ++e) dst[ct + T * e] = (v[e].x * v[e].x + v[e].y * v[e].y) * g.scale;
            }
            // the buffer tile k + 2 lands in is this one: every thread of the team must be past its exchanges
            if (mode != 0) sm.sync();
        }
    };

    auto load_lines = [&](float2 (&v)[E], int y) {
        const float2* row = psi + (size_t)y * N + rt;
#pragma unroll
        for (int e = 0; e < E; ++e) v[e] = x_in_band(e) ? __ldcg(row + T * e) : make_float2(0.f, 0.f);
    };
    // IFFT_x . t_s . FFT_x on every row (Eq. 1 between the transforms)
    auto row_pass = [&](const float2* ts) {
        float2 v[E], vn[E];
#pragma unroll
        for (int e = 0; e < E; ++e) vn[e] = make_float2(0.f, 0.f);
        load_lines(v, rl);
#pragma unroll 1
        for (int y = rl; y < N; y += C::LINES) {
            if (y + C::LINES < N) load_lines(vn, y + C::LINES);
            fft_inverse<P>(v, twr, rt, rsm);
            const float2* trow = ts + (size_t)y * N + rt;
#pragma unroll
            for (int e = 0; e < E; ++e) v[e] = cmul(v[e], __ldg(trow + T * e));
            fft_forward<P>(v, twr, rt, rsm);
            float2* row = psi + (size_t)y * N + rt;
#pragma unroll
            for (int e = 0; e < E; ++e)
                if (x_in_band(e)) row[T * e] = v[e];
#pragma unroll
            for (int e = 0; e < E; ++e) v[e] = vn[e];
        }
    };

    for (int probe = g.probe0 + blockIdx.x; probe < g.probe0 + g.n_probes; probe += gridDim.x) {
        column_pass(0, probe);
        __syncthreads();
        for (int s = 0; s < g.n_slices; ++s) {
            row_pass(g.t_stack + (size_t)s * N * N);
            __syncthreads();
            column_pass(s + 1 < g.n_slices ? 1 : 2, probe);
            __syncthreads();
        }
        // annular rings: one warp per ring, host-built pixel lists, fixed order
        for (int b = warp; b < g.n_bins; b += C::THREADS / 32) {
            const int lo = __ldg(g.bin_start + b), hi = __ldg(g.bin_start + b + 1);
            float sum = 0.f;
            for (int i = lo + lane; i < hi; i += 32) sum += __ldcg(inten + __ldg(g.bin_pix + i));
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
            if (lane == 0) g.out[(size_t)probe * g.n_bins + b] = sum;
        }
        __syncthreads();                                     // the next probe's last pass rewrites the intensity slot
    }
}

template <int N, int XBE, int YBE>
static cudaError_t launch_ms_t(const MsResidentArgs& g, cudaStream_t stream)
{
    using C = MsCfg<N>;
    auto kern = ms_resident_kernel<N, XBE, YBE>;
    static PerDevice once{};
    if (cudaError_t e = opt_in_smem(kern, C::SMEM, once); e != cudaSuccess) return e;
    int grid = g.n_probes < g.slots ? g.n_probes : g.slots;
    if (grid > num_sms()) grid = num_sms();
    kern<<<grid, C::THREADS, C::SMEM, stream>>>(g);
    return cudaGetLastError();
}

template <int N>
static cudaError_t launch_ms_n(const MsResidentArgs& g, cudaStream_t stream)
{
    using C = MsCfg<N>;
    constexpr int XB = DefaultBand<N>::XB;
    if (g.xband % C::W || 2 * g.xband > N) return cudaErrorInvalidValue;
    if constexpr (XB % C::T == 0)
        if (g.xband == XB && g.yband == XB) return launch_ms_t<N, XB / C::T, XB / C::T>(g, stream);
    return launch_ms_t<N, 0, 0>(g, stream);
}

cudaError_t launch_ms_resident(const MsResidentArgs& g, cudaStream_t stream)
{
    if (g.n_probes <= 0) return cudaSuccess;
    switch (g.n) {
        case 256: return launch_ms_n<256>(g, stream);
        case 512: return launch_ms_n<512>(g, stream);
    }
    return cudaErrorInvalidValue;
}

}  // namespace prism
