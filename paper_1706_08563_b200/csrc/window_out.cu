// window_out.cu -- PRISM stage 2 after the beam sum, fused: the summed probe window stays on chip from its one
// read to the ring sums.
//
// PAPER.md:128 "the modulus squared of its FFT ... is integrated" ; "an array of annular ring virtual
// detectors" ; SURVEY.md rows S2-c / S2-d ("M x M complex64 in shared memory", "kept on-chip").
//
// One CTA per window w[my][mx] (complex64, up to 128 x 128 = 128 KB), persistent over the windows of a batch:
//   (1) row pass    : every line goes from HBM straight into registers (8-byte coalesced loads, the next pass's
//                     lines are requested before the current ones are transformed and stay in registers across
//                     the other phases), FFT_x with the line's own shared-memory row as exchange space, result
//                     left in that row;
//   (2) column pass : FFT_y of every column in registers (the column's own storage is the exchange space),
//                     I = |.|^2 / (mx my) written into the real part of the same slots (and, when the caller wants
//                     patterns or mask detectors, to HBM with ky contiguous);
//   (3) rings       : one warp per ring walks the host-built (fp64) pixel list of the ring -- kept in shared memory
//                     as 16-bit tile offsets for the whole launch -- in a fixed order: deterministic sums.
// HBM traffic per probe: one read of the window (8 mx my bytes) and n_bins floats out.
// The transforms and the summation order are those of row_pass_kernel / col_pass_kernel / bin_reduce_kernel
// (slice_pass.cu, output.cu), which this kernel replaces on the PRISM output path.
// complex adds of the register butterflies as packed FADD2: the kernel is bound by issue slots (16 warps per SM)
#define PRISM_PACKED_ADDS 1
#include "fft_core.cuh"
#include "prism_internal.h"

namespace prism {

template <int MX, int MY>
struct WinCfg {
    using PX = typename PlanFor<MX>::type;
    using PY = typename PlanFor<MY>::type;
    static constexpr int TX = PX::T, TY = PY::T, EX = PX::E, EY = PY::E;
    static constexpr int CS = PX::PADDED | 1;                    // row stride of the tile (odd, >= padded line)
    static constexpr int ROWS = PY::PADDED;                      // padded row index space
    static constexpr int WANT = (MY * TX < MX * TY) ? MY * TX : MX * TY;
    static constexpr int NT = WANT < 512 ? (WANT < 32 ? 32 : WANT) : 512;
    static constexpr int LR = NT / TX, LC = NT / TY;             // lines per row pass / column pass
    static constexpr int RP = (MY + LR - 1) / LR, CP = (MX + LC - 1) / LC;
    static constexpr size_t TILE_BYTES = (size_t)ROWS * CS * sizeof(float2);
    static constexpr int TWX = SmemTwiddles<PX>::COUNT, TWY = SmemTwiddles<PY>::COUNT;      // inter-stage twiddles (float2)
    static constexpr size_t FIXED_BYTES = (TILE_BYTES + (size_t)(TWX + TWY) * sizeof(float2) + 15) / 16 * 16;
    static_assert(ROWS * CS < 65536, "tile offsets must fit 16 bits");
};

template <int MX, int MY>
__global__ void __launch_bounds__(WinCfg<MX, MY>::NT) window_out_kernel(WindowArgs g)
{
    using C = WinCfg<MX, MY>;
    using PX = typename C::PX;
    using PY = typename C::PY;
    constexpr int TX = C::TX, TY = C::TY, EX = C::EX, EY = C::EY, CS = C::CS, NT = C::NT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* tile = reinterpret_cast<float2*>(smem_raw);                                   // [ROWS][CS]
    float2* twtab = reinterpret_cast<float2*>(smem_raw + C::TILE_BYTES);                  // [TWX + TWY]
    int* ring_start = reinterpret_cast<int*>(smem_raw + C::FIXED_BYTES);                  // [n_bins + 1]
    unsigned short* ring_off = reinterpret_cast<unsigned short*>(ring_start + ((g.n_bins + 1 + 3) & ~3));   // [listed pixels]
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    // ring lists: pixel kx * MY + ky of the (transposed) pattern -> offset of its slot in the tile
    const int n_listed = g.out ? __ldg(g.bin_start + g.n_bins) : 0;
    if (g.out) {
        for (int i = tid; i <= g.n_bins; i += NT) ring_start[i] = __ldg(g.bin_start + i);
        for (int i = tid; i < n_listed; i += NT) {
            const int pix = __ldg(g.bin_pix + i);
            const int kx = pix / MY, ky = pix % MY;
            ring_off[i] = (unsigned short)(pad16(ky) * CS + pad16(kx));
        }
    }
    const int lx = tid / TX, tx = tid % TX;           // row pass: line of the pass, thread of the line
    const int ly = tid / TY, ty = tid % TY;           // column pass
    SmemTwiddles<PX>::fill(twtab, g.tw_x, tid, NT);
    SmemTwiddles<PY>::fill(twtab + C::TWX, g.tw_y, tid, NT);
    __syncthreads();
    SmemTwiddles<PX> twx;
    twx.bind(twtab, tx);
    SmemTwiddles<PY> twy;
    twy.bind(twtab + C::TWX, ty);

    const size_t npix = (size_t)MX * MY;
    auto load_rows = [&](float2 (&v)[EX], long long win, int pass) {
        if (win >= g.n) return;
        int row = pass * C::LR + lx;
        if (row >= MY) row = MY - 1;
        const float2* src = g.w + (size_t)win * npix + (size_t)row * MX + tx;
#pragma unroll
        for (int e = 0; e < EX; ++e) v[e] = __ldg(src + TX * e);
    };

    float2 cur[EX], nxt[EX];
#pragma unroll
    for (int e = 0; e < EX; ++e) cur[e] = nxt[e] = make_float2(0.f, 0.f);
    load_rows(cur, blockIdx.x, 0);
    for (long long win = blockIdx.x; win < g.n; win += gridDim.x) {
        // ---- (1) FFT_x of every row, in place in the tile ----
#pragma unroll
        for (int pass = 0; pass < C::RP; ++pass) {
            if (pass + 1 < C::RP) load_rows(nxt, win, pass + 1);
            else load_rows(nxt, win + gridDim.x, 0);
            const int row = pass * C::LR + lx;
            const bool active = row < MY;
            const LineSmem<PX> sm{ tile + pad16(active ? row : MY - 1) * CS, 1 };
            if (active || C::LR * C::RP == MY) {
                fft_forward<PX>(cur, twx, tx, sm);
                sm.sync();                            // the other threads of the line are done with the exchange
#pragma unroll
                for (int e = 0; e < EX; ++e) sm.st(tx + TX * e, cur[e]);
            }
#pragma unroll
            for (int e = 0; e < EX; ++e) cur[e] = nxt[e];
        }
        __syncthreads();

        // ---- (2) FFT_y of every column, |.|^2 / (mx my) into the real part of the column's own slots ----
#pragma unroll
        for (int pass = 0; pass < C::CP; ++pass) {
            const int c = pass * C::LC + ly;
            if (c < MX || C::LC * C::CP == MX) {
                const LineSmem<PY> sm{ tile + pad16(c), CS };
                float2 v[EY];
#pragma unroll
                for (int e = 0; e < EY; ++e) v[e] = sm.ld(ty + TY * e);
                fft_forward<PY>(v, twy, ty, sm);
                sm.sync();
#pragma unroll
                for (int e = 0; e < EY; ++e) {
                    const float inten = (v[e].x * v[e].x + v[e].y * v[e].y) * g.scale;
                    tile[pad16(ty + TY * e) * CS + pad16(c)].x = inten;
                    if (g.intensity) g.intensity[(size_t)win * npix + (size_t)c * MY + ty + TY * e] = inten;
                }
            }
        }
        __syncthreads();

        // ---- (3) annular rings: one warp per ring, fixed order ----
        if (g.out) {
            const float* tf = reinterpret_cast<const float*>(tile);
            for (int b = warp; b < g.n_bins; b += NT / 32) {
                const int lo = ring_start[b], hi = ring_start[b + 1];
                float sum = 0.f;
                for (int i = lo + lane; i < hi; i += 32) sum += tf[2 * (int)ring_off[i]];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
                if (lane == 0) g.out[(size_t)win * g.n_bins + b] = sum;
            }
            __syncthreads();                          // the tile is rewritten by the next window's rows
        }
    }
}

template <int MX, int MY>
static cudaError_t launch_window_t(const WindowArgs& g, cudaStream_t stream)
{
    using C = WinCfg<MX, MY>;
    auto kern = window_out_kernel<MX, MY>;
    const size_t lists = g.out ? (size_t)((g.n_bins + 1 + 3) & ~3) * sizeof(int) + (size_t)MX * MY * sizeof(unsigned short) : 16;
    const size_t smem = C::FIXED_BYTES + lists;
    if (smem > 227 * 1024) return cudaErrorInvalidValue;
    // the ring lists make the shared-memory size depend on n_bins: opt in to the largest size once, occupancy per size
    static PerDevice once{};
    if (cudaError_t e = opt_in_smem(kern, 227 * 1024, once); e != cudaSuccess) return e;
    int per_sm = 0;
    if (cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, C::NT, smem); e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorInvalidValue;
    long long grid = (long long)num_sms() * per_sm;
    if (grid > g.n) grid = g.n;
    kern<<<(unsigned)grid, C::NT, smem, stream>>>(g);
    return cudaGetLastError();
}

template <int MX>
static cudaError_t launch_window_x(const WindowArgs& g, cudaStream_t stream)
{
    switch (g.my) {
        case 16:  return launch_window_t<MX, 16>(g, stream);
        case 32:  return launch_window_t<MX, 32>(g, stream);
        case 64:  return launch_window_t<MX, 64>(g, stream);
        case 128: if constexpr (MX * 128 <= 128 * 128) return launch_window_t<MX, 128>(g, stream); else break;
    }
    return cudaErrorInvalidValue;
}

cudaError_t launch_window_out(const WindowArgs& g, cudaStream_t stream)
{
    if (g.n <= 0) return cudaSuccess;
    if (!g.out && !g.intensity) return cudaErrorInvalidValue;
    switch (g.mx) {
        case 16:  return launch_window_x<16>(g, stream);
        case 32:  return launch_window_x<32>(g, stream);
        case 64:  return launch_window_x<64>(g, stream);
        case 128: return launch_window_x<128>(g, stream);
    }
    return cudaErrorInvalidValue;
}

}  // namespace prism
