// prism_internal.h -- declarations shared by the translation units of
// libprism_b200.so (not part of the public C ABI, see include/prism.h).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include <atomic>

namespace prism {

// ---- per-device launch set-up -----------------------------------------------------
// Function attributes (the opt-in to more than 48 KiB of dynamic shared memory) and occupancy results belong to
// a device, so "already done" is remembered per device.  The marks are idempotent: two host threads racing on the
// same mark both do the (identical) set-up.
constexpr int MAX_DEVICES = 64;
inline int current_device()
{
    int d = 0;
    if (cudaGetDevice(&d) != cudaSuccess || d < 0 || d >= MAX_DEVICES) d = 0;
    return d;
}
struct PerDevice { std::atomic<int> v[MAX_DEVICES]; };
template <class K>
inline cudaError_t opt_in_smem(K kern, size_t smem, PerDevice& once)
{
    const int d = current_device();
    if (once.v[d].load(std::memory_order_acquire)) return cudaSuccess;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    once.v[d].store(1, std::memory_order_release);
    return cudaSuccess;
}
// resident CTAs per SM of `kern` at this launch shape on the current device (after the shared-memory opt-in)
template <class K>
inline int blocks_per_sm_cached(K kern, int threads, size_t smem, PerDevice& cache)
{
    const int d = current_device();
    int n = cache.v[d].load(std::memory_order_acquire);
    if (n > 0) return n;
    if (smem > 48 * 1024) cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    n = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, threads, smem);
    if (n <= 0) n = 1;
    cache.v[d].store(n, std::memory_order_release);
    return n;
}

// ---- slice-step passes (slice_pass.cu) -----------------------------------------
// Waves live in "mixed space" A[w][y][kx] = sum_x psi[w][y][x] exp(-2 pi i kx x / nx)
// between the two passes of a slice.
enum RowMode {
    ROW_INIT  = 0,   // plane wave b  -> * t            -> FFT_x -> A          (first slice, no read)
    ROW_STEP  = 1,   // A -> IFFT_x   -> * t            -> FFT_x -> A
    ROW_FINAL = 2,   // A -> IFFT_x   -> * scale        -> out   (real-space exit wave, S-matrix layer)
};
struct RowArgs {
    float2*       a;          // [n_waves][ny][nx] in/out
    float2*       out;        // ROW_FINAL destination (may alias a)
    const float2* t;          // [ny][nx] transmission function of this slice (ROW_INIT, ROW_STEP)
    const float2* tw_x;       // exp(-2 pi i m / nx), m < nx
    const float2* tw_y;       // exp(-2 pi i m / ny), m < ny   (ROW_INIT phase of the plane wave)
    const int2*   beams;      // [n_waves] (kx, ky)             (ROW_INIT)
    int           n_waves, nx, ny;
    int           xband;      // mixed space is read / written for kx in [0, xband) and [nx - xband, nx) only
                              // (pipelined kernels; everything outside is zero by the 2/3 band-limit)
    int           blocked;    // 1: mixed space in the blocked layout "B8" (blocked_grid(); slice_pk.cu); ROW_FINAL then
                              // needs out != a (real space is natural order: the layouts differ, no in-place pass)
    float         scale;      // ROW_INIT: plane-wave amplitude; ROW_FINAL: output scale
};
cudaError_t launch_row_pass(RowMode mode, const RowArgs& args, cudaStream_t stream);
// grids whose slice step runs on the pipelined kernels of slice_pipe_row.cu / slice_pipe_col.cu or the packed ones of slice_pk.cu
inline bool pipelined_grid(int nx, int ny) { return nx >= 256 && ny >= 256; }
cudaError_t launch_row_pipe(RowMode mode, const RowArgs& args, cudaStream_t stream);
// line lengths whose row pass runs on the packed-FFT kernels of slice_pk.cu; their transmission function is
// stored in pair layout t[y][j] = (re(2j), re(2j+1), im(2j), im(2j+1))
inline bool packed_row(int nx, int ny) { return pipelined_grid(nx, ny) && nx == 2048; }
cudaError_t launch_row_pk(RowMode mode, const RowArgs& args, cudaStream_t stream);
// grids whose mixed space uses the blocked layout "B8" (slice_pk.cu): tiles of 8 in-band columns, each tile
// [ny][8] contiguous, so that the 2048-point column pass moves 128 KB runs instead of 32-byte row segments
#ifndef PRISM_BLOCKED_LAYOUT
#define PRISM_BLOCKED_LAYOUT 1
#endif
inline bool blocked_grid(int nx, int ny) { return PRISM_BLOCKED_LAYOUT && nx == 2048 && ny == 2048; }

enum ColMode {
    COL_STEP     = 0,   // A -> FFT_y -> * P -> IFFT_y -> A
    COL_MS_INIT  = 1,   // probe spectrum Psi0(kx, ky) -> IFFT_y -> A          (multislice start, no read)
    COL_MS_FINAL = 2,   // A -> FFT_y -> * P -> |.|^2 -> intensity[w][kx][ky]  (multislice end, no IFFT)
};
struct ColArgs {
    float2*       a;          // [n_waves][ny][nx] in/out
    float*        intensity;  // [n_waves][nx][ny]  (COL_MS_FINAL) -- transposed: ky contiguous
    const float2* tw_y;       // exp(-2 pi i m / ny)
    const float2* prop_x;     // [nx] x-factor of the propagator (all scale factors folded in)
    const float2* prop_y;     // [ny] y-factor
    const int*    ky_lim;     // [nx] band-limit: |ky| <= ky_lim[kx] passes, -1 = whole column masked
    // COL_MS_INIT
    const float2* aperture_t; // [nx][ny] A_k exp(-i chi_k) * amplitude (transposed, ky contiguous)
    const float2* phase_x;    // [probes_x][nx] exp(-2 pi i kx x_p / lx)
    const float2* phase_y;    // [probes_y][ny] exp(-2 pi i ky y_p / ly)
    int           probe0, probes_x;   // wave w is probe probe0 + w; (px, py) = (p % probes_x, p / probes_x)
    int           n_waves, nx, ny;
    int           xband;      // see RowArgs
    int           yband;      // a multiple of 32 with ky_lim[kx] < yband for every kx (pipelined kernels)
    int           blocked;    // 1: mixed space in the blocked layout "B8" (see RowArgs)
    float         scale;      // COL_MS_FINAL intensity scale
};
cudaError_t launch_col_pass(ColMode mode, const ColArgs& args, cudaStream_t stream);
cudaError_t launch_col_pipe(ColMode mode, const ColArgs& args, cudaStream_t stream);
// column lengths whose column pass runs on the packed-FFT kernels of slice_pk.cu
inline bool packed_col(int nx, int ny) { return pipelined_grid(nx, ny) && ny == 2048; }
cudaError_t launch_col_pk(ColMode mode, const ColArgs& args, cudaStream_t stream);

// Resident multislice (ms_resident.cu): one launch carries probes probe0 .. probe0 + n_probes - 1 through all slices,
// one probe per CTA at a time, from the probe spectrum to the ring sums.  Square grids of 256 or 512 points whose
// transmission functions of all slices are in device memory.
struct MsResidentArgs {
    float2*       psi;        // [slots][n][n] wave storage, one slot per CTA
    float*        intensity;  // [slots][n][n] detector plane, transposed (ky contiguous); out-of-band columns stay zero
    const float2* t_stack;    // [n_slices][n][n] transmission functions
    const float2* tw;         // exp(-2 pi i m / n)
    const float2* prop_x;     // see ColArgs
    const float2* prop_y;
    const int*    ky_lim;
    const float2* aperture_t; // [n][n] A_k exp(-i chi_k) * amplitude (transposed)
    const float2* phase_x;    // [probes_x][n]
    const float2* phase_y;    // [probes_y][n]
    const int*    bin_start;  // ring lists over pixel index kx * n + ky
    const int*    bin_pix;
    float*        out;        // [all probes][n_bins]
    int           n, n_slices, probe0, n_probes, probes_x, n_bins, xband, yband, slots;
    float         scale;      // intensity scale of the last column pass
};
inline bool resident_grid(int nx, int ny) { return nx == ny && (nx == 256 || nx == 512); }
constexpr int RESIDENT_SLOTS = 148;   // waves in flight: one per SM of a B200
cudaError_t launch_ms_resident(const MsResidentArgs& args, cudaStream_t stream);

// t = exp(i sigma V) for one slice (Eq. 1), fp64 sincos rounded once to fp32
cudaError_t launch_transmission(const float* v, float2* t, double sigma, int64_t npix, bool pairs, cudaStream_t stream);

// ---- stage 2 (output.cu) ---------------------------------------------------------
struct BeamSumArgs {
    const float2* s;          // [n_beams][ny][nx] compact S-matrix
    float2*       w;          // [n_probes_batch][my][mx] summed windows (out)
    const float2* coef_b;     // [n_beams]  A_b exp(-i chi_b) * scale
    const float2* phase_x;    // [probes_x][n_beams] exp(-2 pi i kx_b x_p / lx)
    const float2* phase_y;    // [probes_y][n_beams] exp(-2 pi i ky_b y_p / ly)
    const int*    win_x0;     // [probes_x] first window column (already wrapped into [0, nx))
    const int*    win_y0;     // [probes_y] first window row
    int           n_beams, nx, ny, mx, my;
    int           probe0, n_probes_batch, probes_x;
};
cudaError_t launch_beam_sum(const BeamSumArgs& args, cudaStream_t stream);

// Regular probe lattice (probe step = 2^k pixels dividing the window): for one S-matrix pixel the
// probe phases exp(-2 pi i q_b . r_p) over the probe lattice are a Q x Q DFT over the beam lattice
// (Q = window / step), so all Q^2 probes whose windows hold that pixel are served by one small
// 2-D FFT instead of Q^2 separate beam sums (same sums, reordered).
struct LatticeArgs {
    const float2* s;          // [n_beams][ny][nx] compact S-matrix
    float2*       w;          // [n_rows * probes_x][my][mx] summed windows of the batch (out)
    const float2* coef;       // [n_beams] A_b exp(-i chi_b) * scale * exp(-2 pi i q_b . r_probe0)
    const int*    cell_beam;  // [n_slots][q * q]: beams folded onto lattice residue (ky/f mod q, kx/f mod q); -1 = none
    int           n_slots, q;
    int           nx, ny, mx, my;
    int           sx_log2, sy_log2;   // probe step in pixels = 1 << s_log2
    int           x00, y00;           // window origin of probe (0, 0), wrapped
    int           probes_x, probes_y;
    int           py0, n_rows;        // probe rows [py0, py0 + n_rows) of this batch
    int           row0, n_pix_rows;   // pixel rows y' = (row0 + r) mod ny, r < n_pix_rows, y' relative to y00
    int           slab;               // 1: s is a ring of pixel rows [n_beams][slab_cap][nx] (S in host memory): row r of
                                      // the batch sits at ring row (slab_u0 + r) % slab_cap of every layer
    int           slab_cap, slab_u0;
};
cudaError_t launch_lattice_dft(const LatticeArgs& args, cudaStream_t stream);

// out[w][bin] = sum of intensity[w][pix] over the pixels listed for the bin (CSR), fixed order
cudaError_t launch_bin_reduce(const float* intensity, int64_t npix, const int* bin_start,
                              const int* bin_pix, int n_bins, float* out, int n_waves,
                              cudaStream_t stream);

// Fused stage-2 epilogue (window_out.cu): FFT2 of every summed window, |.|^2 * scale, ring sums -- the window is read
// once and stays in shared memory.  `out` and / or `intensity` may be null (but not both).
struct WindowArgs {
    const float2* w;          // [n][my][mx] summed windows
    const float2* tw_x;       // exp(-2 pi i m / mx)
    const float2* tw_y;       // exp(-2 pi i m / my)
    const int*    bin_start;  // [n_bins + 1] CSR ring lists over pixel index kx * my + ky (host fp64 decisions)
    const int*    bin_pix;
    float*        out;        // [n][n_bins] ring sums
    float*        intensity;  // [n][mx][my] patterns, ky contiguous (for the 4-D output and mask detectors)
    int           n, mx, my, n_bins;
    float         scale;      // 1 / (mx my)
};
cudaError_t launch_window_out(const WindowArgs& args, cudaStream_t stream);

// patterns[w][ky][kx] = intensity[w][kx][ky]: the column pass writes patterns transposed (ky contiguous), the 4-D
// output wants them in natural order
cudaError_t launch_transpose_patterns(const float* intensity, float* patterns, int mx, int my, int n_waves,
                                      cudaStream_t stream);

// out[w][d] = sum over pixels of masks[d][ky][kx] * intensity[w][kx][ky], d < n_masks <= 16 (virtual detectors)
cudaError_t launch_mask_dot(const float* intensity, const float* masks, int n_masks, int mx, int my, float* out,
                            int n_waves, cudaStream_t stream);

// acc = (first ? 0 : acc) + weight * x   (frozen-phonon accumulation)
cudaError_t launch_accumulate(float* acc, const float* x, int64_t n, float weight, bool first, cudaStream_t stream);
int num_sms();

// ---- potential (potential.cu) ------------------------------------------------------
struct PotAtom { double x, y; int32_t lut; int32_t pad; };
struct PotentialArgs {
    const PotAtom* atoms;       // sorted by (slice, tile_y, tile_x)
    const int*     cell_start;  // [n_slices * tiles_y * tiles_x + 1]
    const float*   lut_v;       // [n_luts][lut_n]
    const double*  lut_rcut;    // [n_luts]
    int            lut_n;
    int            nx, ny, tiles_x, tiles_y, tile, reach_tiles;
    double         px, py, lx, ly;
    int            slice0, n_slices_chunk;   // slices [slice0, slice0 + n_slices_chunk) -> v_out
    float*         v_out;       // [n_slices_chunk][ny][nx]
};
cudaError_t launch_potential(const PotentialArgs& args, cudaStream_t stream);
// Device address, on the current device, of the library's built-in scratch array of POT_STATIC_BYTES bytes
// (prism_build_potential_static).  The first call on a device looks the address up; no allocation.
constexpr size_t POT_STATIC_BYTES = (size_t)8 << 20;
cudaError_t potential_static_scratch(void** ptr);

}  // namespace prism
