// output.cu -- PRISM stage 2: cropped-window beam sum, and the annular-bin
// reduction shared with plain multislice.
//
// PAPER.md:86  "For each probe, a subset of all plane waves is cut out around the
//   maximum value of the input STEM probe. The size length of the subset regions
//   is d/f ... Each STEM probe is computed by multiplying each plane wave subset by
//   the appropriate coefficient and summing all wave subsets."
// PAPER.md:128 "applying coefficients, one for each plane wave, to the elements of
//   the compact S-matrix and summing along the dimension corresponding to the
//   different plane waves ... coefficients ... precomputed ... read ... into
//   shared memory".
// PAPER.md:82  "an array of annular ring virtual detectors".
#include "fft_core.cuh"
#include "prism_internal.h"

namespace prism {

// One CTA per probe.  Coefficients c_b = coef_b * phase_x[px][b] * phase_y[py][b]
// are formed once in shared memory; every thread owns PPT window pixels and runs
// over the beams with PPT independent coalesced 8-byte loads in flight.
constexpr int BEAM_SUM_PPT = 16;

template <int PPT>
__global__ void __launch_bounds__(1024) beam_sum_kernel(BeamSumArgs g)
{
    extern __shared__ float2 coef[];                 // [n_beams]
    const int p = g.probe0 + blockIdx.x;
    const int pxi = p % g.probes_x, pyi = p / g.probes_x;
    for (int b = threadIdx.x; b < g.n_beams; b += blockDim.x) {
        const float2 ex = __ldg(g.phase_x + (size_t)pxi * g.n_beams + b);
        const float2 ey = __ldg(g.phase_y + (size_t)pyi * g.n_beams + b);
        coef[b] = cmul(cmul(__ldg(g.coef_b + b), ex), ey);
    }
    __syncthreads();

    const int npix = g.mx * g.my;
    const int x0 = g.win_x0[pxi], y0 = g.win_y0[pyi];
    int off[PPT];                                     // offset of each owned pixel inside one S layer
#pragma unroll
    for (int e = 0; e < PPT; ++e) {
        int q = threadIdx.x + e * blockDim.x;
        if (q >= npix) q = npix - 1;
        const int j = q / g.mx, i = q % g.mx;
        const int yy = (y0 + j) & (g.ny - 1), xx = (x0 + i) & (g.nx - 1);
        off[e] = yy * g.nx + xx;
    }
    float2 acc[PPT];
#pragma unroll
    for (int e = 0; e < PPT; ++e) acc[e] = make_float2(0.f, 0.f);

    const size_t layer = (size_t)g.nx * g.ny;
    const float2* s = g.s;
    for (int b = 0; b < g.n_beams; ++b, s += layer) {
        const float2 c = coef[b];
        float2 val[PPT];
#pragma unroll
        for (int e = 0; e < PPT; ++e) val[e] = __ldg(s + off[e]);
#pragma unroll
        for (int e = 0; e < PPT; ++e) {
            acc[e].x = fmaf(c.x, val[e].x, acc[e].x); acc[e].x = fmaf(-c.y, val[e].y, acc[e].x);
            acc[e].y = fmaf(c.x, val[e].y, acc[e].y); acc[e].y = fmaf(c.y, val[e].x, acc[e].y);
        }
    }
    float2* wout = g.w + (size_t)blockIdx.x * npix;
#pragma unroll
    for (int e = 0; e < PPT; ++e) {
        const int q = threadIdx.x + e * blockDim.x;
        if (q < npix) wout[q] = acc[e];
    }
}

cudaError_t launch_beam_sum(const BeamSumArgs& g, cudaStream_t stream)
{
    if (g.n_probes_batch == 0) return cudaSuccess;
    const int npix = g.mx * g.my;
    int threads = (npix + BEAM_SUM_PPT - 1) / BEAM_SUM_PPT;
    threads = ((threads + 31) / 32) * 32;
    if (threads > 1024) return cudaErrorInvalidValue;       // windows up to 128 x 128
    const size_t smem = (size_t)g.n_beams * sizeof(float2);
    if (smem > 48 * 1024) {
        static bool set = false;
        if (!set) { cudaFuncSetAttribute(beam_sum_kernel<BEAM_SUM_PPT>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024); set = true; }
        if (smem > 200 * 1024) return cudaErrorInvalidValue;
    }
    beam_sum_kernel<BEAM_SUM_PPT><<<g.n_probes_batch, threads, smem, stream>>>(g);
    return cudaGetLastError();
}

// Annular-ring integration: one CTA per wave, one warp per ring at a time; the
// pixels of each ring are listed by the host (fp64 bin decisions), and are summed
// in a fixed order, so the result is deterministic.
__global__ void __launch_bounds__(256) bin_reduce_kernel(const float* __restrict__ intensity, int64_t npix,
                                                         const int* __restrict__ bin_start,
                                                         const int* __restrict__ bin_pix, int n_bins,
                                                         float* __restrict__ out)
{
    const float* img = intensity + (size_t)blockIdx.x * npix;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, n_warps = blockDim.x >> 5;
    for (int b = warp; b < n_bins; b += n_warps) {
        const int lo = bin_start[b], hi = bin_start[b + 1];
        float sum = 0.f;
        for (int i = lo + lane; i < hi; i += 32) sum += img[bin_pix[i]];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
        if (lane == 0) out[(size_t)blockIdx.x * n_bins + b] = sum;
    }
}

cudaError_t launch_bin_reduce(const float* intensity, int64_t npix, const int* bin_start,
                              const int* bin_pix, int n_bins, float* out, int n_waves,
                              cudaStream_t stream)
{
    if (n_waves == 0 || n_bins == 0) return cudaSuccess;
    bin_reduce_kernel<<<n_waves, 256, 0, stream>>>(intensity, npix, bin_start, bin_pix, n_bins, out);
    return cudaGetLastError();
}

}  // namespace prism
