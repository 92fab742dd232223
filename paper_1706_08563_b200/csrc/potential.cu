// potential.cu -- projected-potential builder (subsystem (a)).
//
// PAPER.md:40  "the sample is divided into slices which are used to compute the
//   projected potential ... implemented by using a precomputed lookup table for each
//   atom type"; "the projected potential for each slice is computed ...
//   using the cached potentials" (on CPU threads in the paper, which notes "In
//   principle this step could be GPU accelerated").
//
// B200 design: a GATHER, not a scatter.  The host sorts atoms into (slice, 16x16-pixel
// tile) cells; one CTA owns one tile of one slice and every thread one pixel, which
// sums the table value of every atom of the surrounding cells that lies within
// r_cut, in the fixed sorted order.  No atomics, no memset, one coalesced write per
// pixel, and a bit-reproducible result.  Distances and the cut decision are taken
// in fp64 (the table interpolation too); the sum is rounded once to fp32.
#include <mutex>

#include "prism_internal.h"

namespace prism {

__global__ void __launch_bounds__(256) potential_kernel(PotentialArgs g)
{
    const int tile = g.tile;                        // 16
    const int tx = blockIdx.x % g.tiles_x, ty = blockIdx.x / g.tiles_x;
    const int sl = blockIdx.y;                      // slice within the chunk
    const int s_abs = g.slice0 + sl;
    const int i = tx * tile + (threadIdx.x % tile), j = ty * tile + (threadIdx.x / tile);
    const double xpix = (double)i * g.px, ypix = (double)j * g.py;
    const double hx = 0.5 * g.lx, hy = 0.5 * g.ly;

    const int ndx = min(2 * g.reach_tiles + 1, g.tiles_x), ndy = min(2 * g.reach_tiles + 1, g.tiles_y);
    double sum = 0.0;
    for (int dy = 0; dy < ndy; ++dy) {
        const int cy = ((ty - g.reach_tiles + dy) % g.tiles_y + g.tiles_y) % g.tiles_y;
        for (int dx = 0; dx < ndx; ++dx) {
            const int cx = ((tx - g.reach_tiles + dx) % g.tiles_x + g.tiles_x) % g.tiles_x;
            const int cell = (s_abs * g.tiles_y + cy) * g.tiles_x + cx;
            const int lo = g.cell_start[cell], hi = g.cell_start[cell + 1];
            for (int a = lo; a < hi; ++a) {
                const PotAtom at = g.atoms[a];
                double ddx = xpix - at.x, ddy = ypix - at.y;
                if (ddx > hx) ddx -= g.lx; else if (ddx < -hx) ddx += g.lx;      // nearest periodic image
                if (ddy > hy) ddy -= g.ly; else if (ddy < -hy) ddy += g.ly;
                const double r = sqrt(ddx * ddx + ddy * ddy);
                const double rc = g.lut_rcut[at.lut];
                if (r > rc) continue;
                const float* tab = g.lut_v + (size_t)at.lut * g.lut_n;
                const double u = r / rc * (double)(g.lut_n - 1);
                const int k = (int)floor(u);
                double val;
                if (k >= g.lut_n - 1) val = (double)tab[g.lut_n - 1];
                else {
                    const double f0 = (double)tab[k], f1 = (double)tab[k + 1];
                    val = f0 + (u - (double)k) * (f1 - f0);
                }
                sum += val;
            }
        }
    }
    if (i < g.nx && j < g.ny)
        g.v_out[((size_t)sl * g.ny + j) * g.nx + i] = (float)sum;
}

cudaError_t launch_potential(const PotentialArgs& g, cudaStream_t stream)
{
    if (g.n_slices_chunk <= 0) return cudaSuccess;
    dim3 grid((unsigned)(g.tiles_x * g.tiles_y), (unsigned)g.n_slices_chunk);
    potential_kernel<<<grid, g.tile * g.tile, 0, stream>>>(g);
    return cudaGetLastError();
}

// ---- scratch for prism_build_potential_static -----------------------------------------------------------
// Some hosts of this library may not allocate device memory themselves: a plug-in that runs inside someone
// else's allocator (a framework whose memory pool owns the whole device), a process that has handed every byte
// to another library, or code running between the capture calls of a stream where cudaMalloc is illegal.  For
// them the kernel's scratch (sorted atoms, cell starts, radial tables) lives here, inside the library image:
// every device that loads the library holds these POT_STATIC_BYTES from load until process exit.
//
// Host code must never hand `pot_static_scratch` itself to a kernel: in host code that name is the host-side
// shadow of the symbol, not a device address.  The device address is looked up once per device with
// cudaGetSymbolAddress (below), with that device current, and cached.
static __device__ __align__(256) unsigned char pot_static_scratch[POT_STATIC_BYTES];

cudaError_t potential_static_scratch(void** ptr)
{
    constexpr int MAX_DEVICES = 64;
    static std::mutex mu;
    static void* address[MAX_DEVICES] = {};
    *ptr = nullptr;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!address[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, pot_static_scratch);       // this device's copy of the array
        if (e != cudaSuccess) return e;
        address[dev] = p;
    }
    *ptr = address[dev];
    return cudaSuccess;
}

}  // namespace prism
