// slice_pass.cu -- the two fused HBM passes of one multislice slice step.
//
// PAPER.md:44 Eq. (1)  psi <- psi * exp(i sigma V)          (transmission)
// PAPER.md:80 Eq. (2)  Psi <- Psi * exp(-i pi lambda q^2 t)  (propagation), "done in Fourier space"
// PAPER.md:132 does these as four separate batched kernels / cuFFT calls (six HBM round trips).
// Here a slice is two passes over the wave batch, each one read + one write:
//   row pass    (fixed y ):  IFFT_x -> * t_s[y][x]      -> FFT_x
//   column pass (fixed kx):  FFT_y  -> * P(kx, ky)      -> IFFT_y
// with the wave kept between passes in mixed space A[w][y][kx].  The same two
// kernels also start and finish the plane waves of the S-matrix
// and the probes of plain multislice.  (The PRISM probe windows of
// PAPER.md:128 are transformed by window_out.cu.)
#include "fft_core.cuh"
#include "prism_internal.h"
#include "pipe_ptx.cuh"

namespace prism {

int num_sms()
{
    static PerDevice cache{};
    const int d = current_device();
    int n = cache.v[d].load(std::memory_order_acquire);
    if (n <= 0) {
        cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, d);
        if (n <= 0) n = 148;
        cache.v[d].store(n, std::memory_order_release);
    }
    return n;
}

__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gmem_src)
{
    unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(s), "l"(gmem_src));
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }

// =============================================================================
// Row pass: LPC lines (rows) per CTA pass, T threads per line, data in registers.
// Line order is (y, wave) with the wave index fastest, so CTAs in flight share the
// same rows of t_s in L2/L1.
// =============================================================================
template <class P, int LPC, int MODE>
__global__ void __launch_bounds__(P::T* LPC) row_pass_kernel(RowArgs g)
{
    constexpr int E = P::E, T = P::T, N = P::N;
    extern __shared__ float2 smem[];
    const int ll = threadIdx.x / T, t = threadIdx.x % T;
    LineSmem<P> sm{ smem + ll * P::PADDED, 1 };
    Twiddles<P> tw;
    tw.load(g.tw_x, t);

    const long long n_lines  = (long long)g.n_waves * g.ny;
    const long long n_groups = (n_lines + LPC - 1) / LPC;
    for (long long grp = blockIdx.x; grp < n_groups; grp += gridDim.x) {
        long long line = grp * LPC + ll;
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
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const float2 wx = __ldg(g.tw_x + ((b.x * (t + T * e)) & (N - 1)));
                v[e] = cmul_conj(base, wx);
            }
        } else {
#pragma unroll
            for (int e = 0; e < E; ++e) v[e] = row[t + T * e];
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
            for (int e = 0; e < E; ++e) row[t + T * e] = v[e];
        }
    }
}

template <class P, int LPC, int MODE>
static cudaError_t launch_row_t(const RowArgs& g, cudaStream_t stream)
{
    auto kern = row_pass_kernel<P, LPC, MODE>;
    const int threads = P::T * LPC;
    const size_t smem = (size_t)LPC * P::PADDED * sizeof(float2);
    static PerDevice occupancy{};
    const int blocks_per_sm = blocks_per_sm_cached(kern, threads, smem, occupancy);
    const long long n_lines = (long long)g.n_waves * g.ny;
    const long long n_groups = (n_lines + LPC - 1) / LPC;
    if (n_groups == 0) return cudaSuccess;
    long long grid = (long long)num_sms() * blocks_per_sm;
    if (grid > n_groups) grid = n_groups;
    kern<<<(unsigned)grid, threads, smem, stream>>>(g);
    return cudaGetLastError();
}

template <int N>
static cudaError_t launch_row_n(RowMode mode, const RowArgs& g, cudaStream_t stream)
{
    using P = typename PlanFor<N>::type;
    constexpr int LPC = (P::T >= 128) ? 1 : 128 / P::T;      // 128 threads per CTA
    switch (mode) {
        case ROW_INIT:  return launch_row_t<P, LPC, ROW_INIT>(g, stream);
        case ROW_STEP:  return launch_row_t<P, LPC, ROW_STEP>(g, stream);
        case ROW_FINAL: return launch_row_t<P, LPC, ROW_FINAL>(g, stream);
    }
    return cudaErrorInvalidValue;
}

cudaError_t launch_row_pass(RowMode mode, const RowArgs& g, cudaStream_t stream)
{
    if (packed_row(g.nx, g.ny)) return launch_row_pk(mode, g, stream);
    if (pipelined_grid(g.nx, g.ny)) return launch_row_pipe(mode, g, stream);
    switch (g.nx) {
        case 16:   return launch_row_n<16>(mode, g, stream);
        case 32:   return launch_row_n<32>(mode, g, stream);
        case 64:   return launch_row_n<64>(mode, g, stream);
        case 128:  return launch_row_n<128>(mode, g, stream);
        case 256:  return launch_row_n<256>(mode, g, stream);
        case 512:  return launch_row_n<512>(mode, g, stream);
        case 1024: return launch_row_n<1024>(mode, g, stream);
        case 2048: return launch_row_n<2048>(mode, g, stream);
    }
    return cudaErrorInvalidValue;
}

// =============================================================================
// Column pass: a CTA stages an [ny rows] x [W columns] tile in shared memory (64 B
// per row segment, rows padded so column accesses are conflict free), transforms
// its columns G groups at a time in registers using the tile's own column storage
// as the exchange space, and streams the tile back.
// =============================================================================
template <class P, int W, int G, int MODE>
__global__ void __launch_bounds__((W / G) * P::T) col_pass_kernel(ColArgs g)
{
    constexpr int E = P::E, T = P::T, N = P::N;
    constexpr int CS = W + 1;                    // padded row stride of the tile (float2 units)
    constexpr int NT = (W / G) * T;
    extern __shared__ float2 tile[];             // [P::PADDED][CS]
    const int tid = threadIdx.x;
    const int cl = tid / T, t = tid % T;
    Twiddles<P> tw;
    tw.load(g.tw_y, t);

    const int tiles_per_wave = g.nx / W;
    const long long n_tiles = (long long)g.n_waves * tiles_per_wave;
    for (long long tl = blockIdx.x; tl < n_tiles; tl += gridDim.x) {
        const int w = (int)(tl / tiles_per_wave), kx0 = (int)(tl % tiles_per_wave) * W;
        float2* base = g.a + (size_t)w * g.ny * g.nx + kx0;

        if (MODE != COL_MS_INIT) {
            for (int i = tid; i < N * W; i += NT) {
                const int row = i / W, c = i % W;
                cp_async8(&tile[pad16(row) * CS + c], base + (size_t)row * g.nx + c);
            }
            cp_async_wait_all();
            __syncthreads();
        }

#pragma unroll 1
        for (int grp = 0; grp < G; ++grp) {
            const int c = grp * (W / G) + cl;
            const int kxi = kx0 + c;                               // array slot of this column
            LineSmem<P> sm{ tile + c, CS };
            float2 v[E];

            if (MODE == COL_MS_INIT) {
                // Psi0(kx, ky) = A_k exp(-i chi_k) exp(-2 pi i (kx xp / lx + ky yp / ly))
                const int p = g.probe0 + w;
                const int pxi = p % g.probes_x, pyi = p / g.probes_x;
                const float2 ex = __ldg(g.phase_x + (size_t)pxi * g.nx + kxi);
                const float2* ap = g.aperture_t + (size_t)kxi * N;
                const float2* ey = g.phase_y + (size_t)pyi * N;
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    const int m = t + T * e;
                    v[e] = cmul(cmul(__ldg(ap + m), ex), __ldg(ey + m));
                }
            } else {
#pragma unroll
                for (int e = 0; e < E; ++e) v[e] = sm.ld(t + T * e);
            }

            if (MODE != COL_MS_INIT) fft_forward<P>(v, tw, t, sm);

            if (MODE == COL_STEP || MODE == COL_MS_FINAL) {
                // Fresnel propagator with the 2/3 band-limit (Eq. 2; BASELINE.json)
                const float2 pxv = __ldg(g.prop_x + kxi);
                const int lim = __ldg(g.ky_lim + kxi);
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    const int m = t + T * e;
                    const int ky = m < N / 2 ? m : N - m;           // |ky|
                    const float2 pr = cmul(pxv, __ldg(g.prop_y + m));
                    v[e] = (ky <= lim) ? cmul(v[e], pr) : make_float2(0.f, 0.f);
                }
            }
            if (MODE == COL_STEP || MODE == COL_MS_INIT) {
                fft_inverse<P>(v, tw, t, sm);
#pragma unroll
                for (int e = 0; e < E; ++e) sm.st(t + T * e, v[e]);   // own slots: no hazard
            } else {
                // detector-plane intensity, ky contiguous
                float* dst = g.intensity + ((size_t)w * g.nx + kxi) * N;
#pragma unroll
                for (int e = 0; e < E; ++e)
                    dst[t + T * e] = (v[e].x * v[e].x + v[e].y * v[e].y) * g.scale;
            }
        }

        if (MODE == COL_STEP || MODE == COL_MS_INIT) {
            __syncthreads();
            for (int i = tid; i < N * W; i += NT) {
                const int row = i / W, c = i % W;
                base[(size_t)row * g.nx + c] = tile[pad16(row) * CS + c];
            }
        }
        __syncthreads();                          // tile is reused by the next iteration
    }
}

template <class P, int W, int G, int MODE>
static cudaError_t launch_col_t(const ColArgs& g, cudaStream_t stream)
{
    auto kern = col_pass_kernel<P, W, G, MODE>;
    const int threads = (W / G) * P::T;
    const size_t smem = (size_t)P::PADDED * (W + 1) * sizeof(float2);
    static PerDevice occupancy{};
    const int blocks_per_sm = blocks_per_sm_cached(kern, threads, smem, occupancy);
    const long long n_tiles = (long long)g.n_waves * (g.nx / W);
    if (n_tiles == 0) return cudaSuccess;
    long long grid = (long long)num_sms() * blocks_per_sm;
    if (grid > n_tiles) grid = n_tiles;
    kern<<<(unsigned)grid, threads, smem, stream>>>(g);
    return cudaGetLastError();
}

template <int N>
static cudaError_t launch_col_n(ColMode mode, const ColArgs& g, cudaStream_t stream)
{
    using P = typename PlanFor<N>::type;
    constexpr int W = 8;
    constexpr int G = (N >= 2048) ? 2 : 1;
    switch (mode) {
        case COL_STEP:     return launch_col_t<P, W, G, COL_STEP>(g, stream);
        case COL_MS_INIT:  return launch_col_t<P, W, G, COL_MS_INIT>(g, stream);
        case COL_MS_FINAL: return launch_col_t<P, W, G, COL_MS_FINAL>(g, stream);
    }
    return cudaErrorInvalidValue;
}

cudaError_t launch_col_pass(ColMode mode, const ColArgs& g, cudaStream_t stream)
{
    if (packed_col(g.nx, g.ny)) return launch_col_pk(mode, g, stream);
    if (pipelined_grid(g.nx, g.ny)) return launch_col_pipe(mode, g, stream);
    if (g.nx % 8 != 0) return cudaErrorInvalidValue;
    switch (g.ny) {
        case 16:   return launch_col_n<16>(mode, g, stream);
        case 32:   return launch_col_n<32>(mode, g, stream);
        case 64:   return launch_col_n<64>(mode, g, stream);
        case 128:  return launch_col_n<128>(mode, g, stream);
        case 256:  return launch_col_n<256>(mode, g, stream);
        case 512:  return launch_col_n<512>(mode, g, stream);
        case 1024: return launch_col_n<1024>(mode, g, stream);
        case 2048: return launch_col_n<2048>(mode, g, stream);
    }
    return cudaErrorInvalidValue;
}

// =============================================================================
// Transmission function of one slice, Eq. (1): t = exp(i sigma V).
// Computed once per slice (not per wave) in fp64 and rounded once to fp32.
// =============================================================================
// PAIRS: pixels (2j, 2j+1) are stored as (re, re, im, im), the layout the packed row pass multiplies in.
template <bool PAIRS>
__global__ void transmission_kernel(const float* __restrict__ v, float2* __restrict__ t, double sigma, int64_t npix)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    griddep_wait();                          // part of the slice loop's chain of dependent launches (pipe_ptx.cuh)
    if (PAIRS) {
        for (; i < npix / 2; i += stride) {
            const float2 vv = reinterpret_cast<const float2*>(v)[i];
            double s0, c0, s1, c1;
            sincos(sigma * (double)vv.x, &s0, &c0);
            sincos(sigma * (double)vv.y, &s1, &c1);
            reinterpret_cast<float4*>(t)[i] = make_float4((float)c0, (float)c1, (float)s0, (float)s1);
        }
    } else {
        for (; i < npix; i += stride) {
            double s, c;
            sincos(sigma * (double)v[i], &s, &c);
            t[i] = make_float2((float)c, (float)s);
        }
    }
}

cudaError_t launch_transmission(const float* v, float2* t, double sigma, int64_t npix, bool pairs, cudaStream_t stream)
{
    if (npix == 0) return cudaSuccess;
    const int threads = 256;
    long long blocks = (npix + threads - 1) / threads;
    const long long cap = (long long)num_sms() * 8;
    if (blocks > cap) blocks = cap;
    if (pairs) return launch_pdl(transmission_kernel<true>, (unsigned)blocks, threads, 0, stream, v, t, sigma, npix);
    return launch_pdl(transmission_kernel<false>, (unsigned)blocks, threads, 0, stream, v, t, sigma, npix);
}

}  // namespace prism
