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
    if (smem > 200 * 1024) return cudaErrorInvalidValue;
    static PerDevice once{};
    if (cudaError_t e = opt_in_smem(beam_sum_kernel<BEAM_SUM_PPT>, 200 * 1024, once); e != cudaSuccess) return e;
    beam_sum_kernel<BEAM_SUM_PPT><<<g.n_probes_batch, threads, smem, stream>>>(g);
    return cudaGetLastError();
}

// =============================================================================
// Lattice DFT (regular probe grids).  PAPER.md:86/:128 define probe p's window as
//   w_p[j][i] = sum_b c_b exp(-2 pi i q_b . r_p) S_b[y0_p + j][x0_p + i].
// With r_p = r_0 + (px, py) * step and step = s pixels (s | window M), beam b =
// (f m_b, f n_b) gives exp(-2 pi i (m_b px + n_b py) / Q), Q = M / s: for a fixed
// S-matrix pixel the values needed by ALL probes are the Q x Q forward DFT of the
// beam lattice array G[n][m] = sum_{b folded onto (n, m) mod Q} c'_b S_b[y][x], and
// the pixel lies in the window of exactly one probe per residue class.  One CTA
// takes TP = 8 * 32/Q pixels of a row: (1) gather + fold + scale into shared
// memory with coalesced reads of S, (2) one warp per 32/Q pixels runs the row and
// column FFT_Q in registers (lane = lattice row / column), (3) the results are
// scattered to the windows, contiguous runs of pixels going to the same probe.
// =============================================================================
template <int Q> struct LatticeCfg {
    static constexpr int NW = 8, NT = NW * 32;          // (16 warps on 16 pixels measured slower: 1.93 against 1.60 ms at P8)
    static constexpr int PW = 32 / Q;                 // pixels per warp
    static constexpr int TP = NW * PW;                // pixels per CTA
    static constexpr int RS = Q + 1;                  // padded row stride (complex)
    static constexpr int PS = Q * RS + (Q == 32 ? 2 : 1);   // pixel stride: conflict-free for phases 1 and 3
    static constexpr size_t SMEM = (size_t)TP * PS * sizeof(float2);
};

// MULTI: more than one beam folds onto some residue (n_slots > 1); a separate instantiation, so that its batched loads
// do not cost the single-slot kernel a resident CTA (92 against 80 registers)
template <int Q, bool MULTI>
__global__ void __launch_bounds__(LatticeCfg<Q>::NT, MULTI ? 2 : 3) lattice_dft_kernel(LatticeArgs g)
{
    using C = LatticeCfg<Q>;
    constexpr int TP = C::TP, RS = C::RS, PS = C::PS, CPI = C::NT / TP;   // cells per iteration
    extern __shared__ float2 sm[];                    // [TP][PS]
    const int tid = threadIdx.x;
    const int tiles_x = g.nx / TP;
    const int r = blockIdx.x / tiles_x, xt = (blockIdx.x % tiles_x) * TP;
    const int yp = (g.row0 + r) & (g.ny - 1);         // row relative to the first window origin
    const int y = (yp + g.y00) & (g.ny - 1);
    const int px = tid % TP, c0 = tid / TP;

    // ---- (1) G[n][m] = sum over folded beams of c'_b S_b[y][x] ----
    {
        // g.slab: g.s is a ring of pixel rows (S itself is in host memory): row r of the batch at ring row (u0 + r) % cap
        const size_t layer = g.slab ? (size_t)g.nx * g.slab_cap : (size_t)g.nx * g.ny;
        const float2* src = g.s + (size_t)(g.slab ? (g.slab_u0 + r) % g.slab_cap : y) * g.nx + xt + px;
        float2* dst = sm + px * PS;
        if (!MULTI) {
#pragma unroll 16
            for (int c = c0; c < Q * Q; c += CPI) {
                const int b = __ldg(g.cell_beam + c);
                float2 r = make_float2(0.f, 0.f);           // residues no beam folds onto: no load
                if (b >= 0) r = cmul(__ldg(g.coef + b), __ldg(src + (size_t)b * layer));
                dst[(c / Q) * RS + (c % Q)] = r;
            }
        } else {
#pragma unroll 4
            for (int c = c0; c < Q * Q; c += CPI) {
                // up to four beams fold onto a residue; the loads of a residue's slots are independent (issued together)
                float2 val[4], cf[4];
#pragma unroll
                for (int sl = 0; sl < 4; ++sl) {
                    const int b = sl < g.n_slots ? __ldg(g.cell_beam + sl * Q * Q + c) : -1;
                    cf[sl] = b >= 0 ? __ldg(g.coef + b) : make_float2(0.f, 0.f);
                    val[sl] = b >= 0 ? __ldg(src + (size_t)b * layer) : make_float2(0.f, 0.f);      // empty slot: no load
                }
                float2 acc = make_float2(0.f, 0.f);
#pragma unroll
                for (int sl = 0; sl < 4; ++sl) acc = cadd(acc, cmul(cf[sl], val[sl]));
                dst[(c / Q) * RS + (c % Q)] = acc;
            }
        }
    }
    __syncthreads();

    // ---- (2) Q x Q forward DFT of every pixel's lattice array, in registers ----
    {
        const int warp = tid >> 5, lane = tid & 31;
        const int rr = lane % Q;
        float2* base = sm + (warp * C::PW + lane / Q) * PS;
        float2 v[Q];
#pragma unroll
        for (int m = 0; m < Q; ++m) v[m] = base[rr * RS + m];           // lattice row n = rr
        Dft<Q>::run(v);                                                  // over m -> probe residue in x
#pragma unroll
        for (int m = 0; m < Q; ++m) base[rr * RS + m] = v[m];
        __syncwarp();
#pragma unroll
        for (int n = 0; n < Q; ++n) v[n] = base[n * RS + rr];           // column: residue x = rr
        Dft<Q>::run(v);                                                  // over n -> probe residue in y
        __syncwarp();
#pragma unroll
        for (int n = 0; n < Q; ++n) base[n * RS + rr] = v[n];
    }
    __syncthreads();

    // ---- (3) scatter: residue (ry, rx) of this pixel belongs to the one probe of that class covering it ----
    {
        const int sx = g.sx_log2, sy = g.sy_log2;
        const int xp = (xt + px - g.x00) & (g.nx - 1);
        const int xc = xp >> sx, xin = xp & ((1 << sx) - 1);
        const int yc = yp >> sy, yin = yp & ((1 << sy) - 1);
        const int wrap_x = g.nx >> sx, wrap_y = g.ny >> sy;
        const size_t npix = (size_t)g.mx * g.my;
        const float2* srcp = sm + px * PS;
#pragma unroll 4
        for (int c = c0; c < Q * Q; c += CPI) {
            const int ry = c / Q, rx = c % Q;
            const int u = (xc - rx) & (Q - 1), v = (yc - ry) & (Q - 1);
            int pp = xc - u, pq = yc - v;
            if (pp < 0) pp += wrap_x;
            if (pq < 0) pq += wrap_y;
            const int prow = pq - g.py0;
            if (pp < g.probes_x && prow >= 0 && prow < g.n_rows) {
                const int i = (u << sx) + xin, j = (v << sy) + yin;
                g.w[((size_t)prow * g.probes_x + pp) * npix + (size_t)j * g.mx + i] = srcp[ry * RS + rx];
            }
        }
    }
}

template <int Q>
static cudaError_t launch_lattice_q(const LatticeArgs& g, cudaStream_t stream)
{
    using C = LatticeCfg<Q>;
    static PerDevice once{};
    if (cudaError_t e = opt_in_smem(lattice_dft_kernel<Q, false>, C::SMEM, once); e != cudaSuccess) return e;
    static PerDevice once_multi{};
    if (cudaError_t e = opt_in_smem(lattice_dft_kernel<Q, true>, C::SMEM, once_multi); e != cudaSuccess) return e;
    if (g.nx % C::TP) return cudaErrorInvalidValue;
    const long long blocks = (long long)(g.nx / C::TP) * g.n_pix_rows;
    if (blocks <= 0) return cudaSuccess;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidValue;
    if (g.n_slots > 1) lattice_dft_kernel<Q, true><<<(unsigned)blocks, C::NT, C::SMEM, stream>>>(g);
    else lattice_dft_kernel<Q, false><<<(unsigned)blocks, C::NT, C::SMEM, stream>>>(g);
    return cudaGetLastError();
}

cudaError_t launch_lattice_dft(const LatticeArgs& g, cudaStream_t stream)
{
    switch (g.q) {
        case 8:  return launch_lattice_q<8>(g, stream);
        case 16: return launch_lattice_q<16>(g, stream);
        case 32: return launch_lattice_q<32>(g, stream);
    }
    return cudaErrorInvalidValue;
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


// 4-D output: one pattern per probe in natural order.  32 x 32 tiles through padded shared memory,
// coalesced on both sides.
__global__ void __launch_bounds__(256) transpose_patterns_kernel(const float* __restrict__ in, float* __restrict__ out,
                                                                 int mx, int my)
{
    __shared__ float tile[32][33];
    const size_t npix = (size_t)mx * my;
    const float* src = in + (size_t)blockIdx.z * npix;       // [kx][ky]
    float* dst = out + (size_t)blockIdx.z * npix;            // [ky][kx]
    const int ky0 = blockIdx.x * 32, kx0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;  // 32 x 8
#pragma unroll
    for (int r = ty; r < 32; r += 8) {
        const int kx = kx0 + r, ky = ky0 + tx;
        if (kx < mx && ky < my) tile[r][tx] = src[(size_t)kx * my + ky];
    }
    __syncthreads();
#pragma unroll
    for (int r = ty; r < 32; r += 8) {
        const int ky = ky0 + r, kx = kx0 + tx;
        if (kx < mx && ky < my) dst[(size_t)ky * mx + kx] = tile[tx][r];
    }
}

cudaError_t launch_transpose_patterns(const float* intensity, float* patterns, int mx, int my, int n_waves,
                                      cudaStream_t stream)
{
    if (n_waves == 0) return cudaSuccess;
    for (int w0 = 0; w0 < n_waves; w0 += 65535) {             // gridDim.z limit
        const int nw = n_waves - w0 < 65535 ? n_waves - w0 : 65535;
        const dim3 grid((my + 31) / 32, (mx + 31) / 32, nw);
        transpose_patterns_kernel<<<grid, 256, 0, stream>>>(intensity + (size_t)w0 * mx * my,
                                                            patterns + (size_t)w0 * mx * my, mx, my);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// Arbitrary virtual detectors: out[w][d] = sum_pix masks[d][ky][kx] * intensity[w][kx][ky].  One CTA per
// pattern walks 32 x 32 tiles: the intensity tile is read with ky contiguous, each mask tile with kx contiguous, and
// they meet through a padded shared-memory tile.  Fixed summation order (deterministic).
constexpr int MAX_MASKS = 16;
template <int NM>                                        // NM >= n_masks: accumulators kept in registers
__global__ void __launch_bounds__(256) mask_dot_kernel(const float* __restrict__ intensity, const float* __restrict__ masks,
                                                       int n_masks, int mx, int my, float* __restrict__ out)
{
    __shared__ float tile[32][33];
    __shared__ float part[8][NM];
    const size_t npix = (size_t)mx * my;
    const float* img = intensity + (size_t)blockIdx.x * npix;        // [kx][ky]
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    float acc[NM];
#pragma unroll
    for (int d = 0; d < NM; ++d) acc[d] = 0.f;
    for (int kx0 = 0; kx0 < mx; kx0 += 32)
        for (int ky0 = 0; ky0 < my; ky0 += 32) {
            __syncthreads();
#pragma unroll
            for (int r = ty; r < 32; r += 8) {
                const int kx = kx0 + r, ky = ky0 + tx;
                tile[r][tx] = (kx < mx && ky < my) ? img[(size_t)kx * my + ky] : 0.f;
            }
            __syncthreads();
#pragma unroll
            for (int r = ty; r < 32; r += 8) {
                const int ky = ky0 + r, kx = kx0 + tx;
                if (kx < mx && ky < my) {
                    const float v = tile[tx][r];
#pragma unroll
                    for (int d = 0; d < NM; ++d)
                        if (d < n_masks) acc[d] = fmaf(__ldg(masks + (size_t)d * npix + (size_t)ky * mx + kx), v, acc[d]);
                }
            }
        }
#pragma unroll
    for (int d = 0; d < NM; ++d) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc[d] += __shfl_xor_sync(0xffffffffu, acc[d], o);
        if (tx == 0) part[ty][d] = acc[d];
    }
    __syncthreads();
    if (threadIdx.x < n_masks) {
        float sum = 0.f;
#pragma unroll
        for (int w = 0; w < 8; ++w) sum += part[w][threadIdx.x];
        out[(size_t)blockIdx.x * n_masks + threadIdx.x] = sum;
    }
}

cudaError_t launch_mask_dot(const float* intensity, const float* masks, int n_masks, int mx, int my, float* out,
                            int n_waves, cudaStream_t stream)
{
    if (n_waves == 0 || n_masks == 0) return cudaSuccess;
    if (n_masks > MAX_MASKS) return cudaErrorInvalidValue;
    if (n_masks <= 1)      mask_dot_kernel<1><<<n_waves, 256, 0, stream>>>(intensity, masks, n_masks, mx, my, out);
    else if (n_masks <= 2) mask_dot_kernel<2><<<n_waves, 256, 0, stream>>>(intensity, masks, n_masks, mx, my, out);
    else if (n_masks <= 4) mask_dot_kernel<4><<<n_waves, 256, 0, stream>>>(intensity, masks, n_masks, mx, my, out);
    else if (n_masks <= 8) mask_dot_kernel<8><<<n_waves, 256, 0, stream>>>(intensity, masks, n_masks, mx, my, out);
    else                   mask_dot_kernel<16><<<n_waves, 256, 0, stream>>>(intensity, masks, n_masks, mx, my, out);
    return cudaGetLastError();
}

// Frozen-phonon accumulation: acc = (first ? 0 : acc) + weight * x, element by element.
__global__ void __launch_bounds__(256) accumulate_kernel(float* __restrict__ acc, const float* __restrict__ x,
                                                         int64_t n, float weight, int first)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
        acc[i] = first ? weight * x[i] : fmaf(weight, x[i], acc[i]);
}

cudaError_t launch_accumulate(float* acc, const float* x, int64_t n, float weight, bool first, cudaStream_t stream)
{
    if (n <= 0) return cudaSuccess;
    long long blocks = (n + 255) / 256;
    const long long cap = (long long)num_sms() * 8;
    if (blocks > cap) blocks = cap;
    accumulate_kernel<<<(unsigned)blocks, 256, 0, stream>>>(acc, x, n, weight, first ? 1 : 0);
    return cudaGetLastError();
}

}  // namespace prism
