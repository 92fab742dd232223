/*
 * prism.h -- C ABI of libprism_b200.so: the data-parallel hot path of PRISM STEM
 * image simulation (arXiv 1706.08563, "Prismatic") on one NVIDIA B200 (sm_100a).
 *
 * Citations are to /root/reference/PAPER.md (line, section/equation) and to the
 * readings R# recorded in DESIGN.md where the paper is silent.
 *
 * Units: lengths in Angstrom, angles in radian, voltage in volt.
 * Arrays are row-major; "[a][b]" means b is contiguous.
 * DFT convention: forward F[k] = sum_n x[n] exp(-2 pi i k n / N), inverse carries
 * 1/N; array slot m holds signed frequency k = m (m < N/2) or m - N.
 *
 * Ownership: the caller owns every buffer (V, S, out, workspace) and the CUDA
 * stream.  The library allocates no device memory ("perform all memory
 * allocations initially") and keeps no simulation state between calls: every call is
 * a function of its arguments.  What it does keep, process-wide, is bookkeeping:
 * per-device marks for one-time kernel set-up (shared-memory opt-in, occupancy), a
 * launch counter, and -- only while prism_timing_enable is on -- a list of timing
 * events (pooled per device: a launch takes its pair from the device current when it
 * is enqueued).  Calls may be made concurrently from several host threads (one per device
 * or stream, the paper's multi-GPU model); the bookkeeping is atomic or
 * mutex-guarded.
 * Work is enqueued on the given stream; outputs are valid once the caller has
 * synchronised that stream.  Host-side tables are built in fp64 inside each call and
 * uploaded from call-local host memory, so each compute call blocks the calling host
 * thread once, until its own table uploads have been consumed (they queue behind work
 * already on the stream); the kernels then run asynchronously.  When a potential or an
 * S-matrix lives in host memory the library moves it over a private copy stream with
 * events, created and released inside the call; all of its copies are joined into
 * `stream`.
 *
 * Errors: every int-returning function returns PRISM_OK (0) or a negative code;
 * nothing aborts, nothing throws across the ABI.  There is no CPU fallback: on a
 * machine without a CUDA device the compute calls return PRISM_ECUDA.
 */
#ifndef PRISM_B200_H
#define PRISM_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    PRISM_OK           =  0,
    PRISM_EINVAL       = -1,  /* null pointer, unsupported grid, f does not divide n, alpha beyond the band-limit, ... */
    PRISM_ENOMEM       = -2,  /* workspace too small (ask prism_workspace_bytes)                                      */
    PRISM_ECUDA        = -3,  /* a CUDA call failed; prism_last_error() holds the CUDA message                        */
    PRISM_EUNSUPPORTED = -4,  /* valid request outside what this build covers (e.g. a window side above 128 points)   */
    PRISM_ENOLUT       = -5   /* an atom's Z has no lookup table                                                     */
};

/* One further term of the aberration function (reading R5b of DESIGN.md; "coherent wave aberrations such
 * as defocus or spherical aberration" are the terms (1,0) and (3,0) of this expansion):
 *   chi(q) += (2 pi / lambda) * c * (lambda |q|)^(n+1) / (n+1) * cos(m (phi - angle)),   phi = atan2(q_y, q_x).
 * c in Angstrom, angle in radian; 1 <= n <= 8, 0 <= m <= n + 1.  Evaluated in fp64 on the host, once per beam
 * (PRISM) or aperture pixel (multislice). */
typedef struct prism_aberration {
    int32_t n, m;
    double  c, angle;
} prism_aberration;

/* The paper's parameters (cell & pixel size PAPER.md:158,:182; slice thickness :158,:200; voltage :182;
 * probe semi-angle :200,:214; interpolation factor f :86; probe grid/step :174,:200; batch_size :126;
 * memory mode :138; annular detectors :82).
 * The struct carries no size or version field: ZERO-INITIALISE it (memset / `= {0}`) and then set what you use, and
 * rebuild callers against this header when it changes.  Fields added later (smatrix_on_host, n_aberrations,
 * aberrations) mean "off" when zero; left uninitialised, n_aberrations / aberrations make the library read through
 * a wild pointer (only the count's range, 0 .. 32, and a NULL pointer can be caught). */
typedef struct prism_params {
    double  cell[3];            /* lx, ly, lz                                                              */
    int32_t nx, ny;             /* grid; pixel = cell / n; powers of two in [64, 2048]                      */
    double  slice_thickness;    /* t of Eq. (2)                                                             */
    int32_t n_slices;           /* S (>= 1); atoms beyond the last slice are clamped into it (R14)          */
    double  voltage;            /* -> lambda, sigma (relativistic closed forms, fp64; R0)                   */
    double  alpha;              /* probe semi-angle; hard aperture edge, '<=' (R4)                          */
    double  defocus, cs;        /* C1, C3: chi(q) = pi lambda q^2 C1 + (pi/2) C3 lambda^3 q^4, probe carries exp(-i chi) (R5) */
    int32_t f;                  /* PRISM interpolation factor; must divide nx and ny; window = n / f (R8);
                                   this build: 16 <= nx / f <= 128 and 16 <= ny / f <= 128, else PRISM_EUNSUPPORTED */
    int32_t probes_x, probes_y; /* probe grid; probe (ix, iy) sits at origin + (ix, iy) * step (R10)         */
    double  probe_origin[2];
    double  probe_step[2];
    double  det_step, det_max;  /* annular ring width and outer angle; n_bins = round(det_max / det_step)    */
    int32_t batch;              /* waves per batch: beams in prism_compute_smatrix, probes in
                                   multislice_compute_output and prism_compute_output; 0 = library default.
                                   Results do not depend on it (PAPER.md:126 batch_size).                   */
    int32_t potential_on_host;  /* 0: V is device memory.  1: V is page-locked host memory and is streamed
                                   slice by slice over a private copy stream.            */
    int32_t smatrix_on_host;    /* 0: S is device memory.  1: S is page-locked host memory ("the
                                   current S-matrix subset": streaming PRISM for S-matrices beyond device memory):
                                   prism_compute_smatrix runs `batch` beams at a time in the workspace and copies
                                   their layers out (copies overlapped with the next batch);
                                   prism_compute_output / _patterns / _detectors keep a ring of pixel rows in the
                                   workspace and bring in the rows the next batch of probe rows adds while the
                                   current one computes (the copies overlap the kernels when consecutive
                                   probe-row batches share or abut pixel rows, i.e. probe-row step <= window
                                   side; otherwise they alternate with them).  Regular probe lattices only. */
    int32_t n_aberrations;      /* further terms of chi beside C1 and C3 (0 .. 32)                           */
    const prism_aberration* aberrations;   /* HOST array of n_aberrations terms (may be NULL when the count is 0) */
} prism_params;

/* Per-species radial table of the projected atomic potential ("precomputed lookup table for
 * each atom type", :116): v[i] = v_Z(r_i), r_i = i * r_cut / (n - 1); v_Z is the piecewise-linear
 * interpolant, 0 beyond r_cut (inclusive cut).  v is HOST memory. */
typedef struct prism_lut {
    int32_t      z;
    int32_t      n;
    double       r_cut;
    const float* v;
} prism_lut;

/* which = */
enum { PRISM_WS_SMATRIX = 0, PRISM_WS_OUTPUT = 1, PRISM_WS_MULTISLICE = 2, PRISM_WS_POTENTIAL = 3,
       PRISM_WS_MULTISLICE_PATTERNS = 4   /* multislice_compute_patterns / _detectors only: they never take the resident
                                             route, so on 256^2 / 512^2 grids they need a batch of waves instead of one
                                             wave per SM (PRISM_WS_MULTISLICE is enough for all three calls, and larger) */
};

/* Bytes of DEVICE workspace the corresponding call needs for these parameters (host-only, no CUDA). */
size_t  prism_workspace_bytes(const prism_params* p, int32_t which);
/* n_bins = round(det_max / det_step) (host-only). */
int32_t prism_num_bins(const prism_params* p);
/* Number of PRISM beams ("every f-th plane wave in both spatial dimensions inside the maximum
 * scattering angle"): signed indices kx = 0 mod f, ky = 0 mod f with (kx/lx)^2 + (ky/ly)^2 <= (alpha/lambda)^2,
 * decided in fp64 on the host. */
int     prism_num_beams(const prism_params* p, int32_t* n_beams);
/* Columns of mixed space A[w][y][kx] that the slice step moves through HBM (host-only): the 2/3 band-limit of
 * the propagator (BASELINE.json; reading R1) leaves kx in [0, c) and [nx - c, nx) only, c = the returned
 * count (a multiple of 32, at most nx / 2), so one pass reads and writes 2 c / nx of a wave.  Grids below
 * 256 points move whole waves (the return value still describes the band). */
int32_t prism_band_columns(const prism_params* p);
/* lambda (Angstrom) and sigma (rad / (V Angstrom)) used by the library for this voltage (host-only). */
int     prism_constants(double voltage, double* lambda, double* sigma);

/* Projected potential (Fig. 1a-b).  For every atom, slice s = clamp(floor(z / t)); every
 * pixel within r_cut of the atom (exact sub-pixel distance, periodic in x and y) receives v_Z(r).
 *   atoms_xyz  HOST  [n_atoms][3] fp64        z_number  HOST [n_atoms]        luts  HOST [n_luts]
 *   v          OUT   [n_slices][ny][nx] fp32: device memory, or page-locked host memory if potential_on_host
 *   workspace  DEVICE, prism_workspace_bytes(p, PRISM_WS_POTENTIAL) + 32 bytes per atom
 * Deterministic (gather, fixed summation order).  Requires 2 r_cut < lx, ly. */
int prism_build_potential(const prism_params* p, const double* atoms_xyz, const int32_t* z_number,
                          int64_t n_atoms, const prism_lut* luts, int32_t n_luts, float* v,
                          void* workspace, size_t workspace_bytes, void* cuda_stream);

/* prism_build_potential for callers that cannot give it a workspace because they may not allocate device memory:
 * code running inside a host application whose own pool owns the device (no cudaMalloc of its own allowed), a
 * process that has already handed all device memory to another library, or a caller inside a phase in which the
 * CUDA allocator must not be entered.  Same arguments, same kernel, same result (bit for bit) as
 * prism_build_potential, minus `workspace`: the scratch the kernel reads (sorted atoms, cell starts, radial
 * tables) is a fixed array of PRISM_STATIC_SCRATCH_BYTES inside the library image.  Every GPU that loads the
 * library carries those bytes from load until the process exits, whether this call is used or not.
 *   Limit: prism_workspace_bytes(p, PRISM_WS_POTENTIAL) + 32 * n_atoms + 512 <= PRISM_STATIC_SCRATCH_BYTES
 *   (configs 1-4 of BASELINE.json fit; config 5's 400 x 2048^2 cell table does not) and potential_on_host = 0
 *   (v is device memory).  Anything beyond returns PRISM_EUNSUPPORTED, with the byte counts in
 *   prism_last_error(); nothing is launched.
 *   The call enters no allocator: no cudaMalloc / cudaFree, no stream or event creation (keep prism_timing_enable
 *   off, which creates events).  Host-side tables are ordinary host memory, as in prism_build_potential.
 *   The first call on each device looks the array's device address up (cudaGetSymbolAddress, with that device
 *   current); make that first call outside any stream capture.
 *   All calls on a device share the one array, and it keeps what the last call left in it.  Every byte the
 *   kernel reads is uploaded on `cuda_stream` by the same call before its launch, so nothing relies on earlier
 *   contents and nothing needs clearing -- but two calls whose GPU work overlaps (different streams or threads,
 *   same device) race on it.  Order them on one stream, or with events. */
#define PRISM_STATIC_SCRATCH_BYTES ((size_t)8 << 20)
int prism_build_potential_static(const prism_params* p, const double* atoms_xyz, const int32_t* z_number,
                                 int64_t n_atoms, const prism_lut* luts, int32_t n_luts, float* v,
                                 void* cuda_stream);

/* Compact S-matrix (Fig. 1g-h): every beam's plane wave exp(+2 pi i q_b . r) is taken
 * through all slices, psi <- IFFT2[ P . FFT2[ psi . exp(i sigma V_s) ] ] (Eq. 1, Eq. 2 with the 2/3
 * band-limit on P), and its real-space exit wave stored as layer b at full resolution (R17).
 *   v      IN   [n_slices][ny][nx] fp32, device or page-locked host (potential_on_host)
 *   beams  OUT  HOST [n_beams][2] int32 (kx, ky) of each layer, n_beams from prism_num_beams
 *   s      OUT  complex64 [n_beams][ny][nx].  smatrix_on_host = 0: DEVICE memory, also the working set (waves are
 *               updated in place).  smatrix_on_host = 1: PAGE-LOCKED HOST memory; `batch` beams at a time are
 *               propagated in the workspace and their layers copied out
 *   workspace DEVICE, prism_workspace_bytes(p, PRISM_WS_SMATRIX) */
int prism_compute_smatrix(const prism_params* p, const float* v, int32_t* beams, void* s,
                          void* workspace, size_t workspace_bytes, void* cuda_stream);

/* PRISM probes (Fig. 1i-k): for every probe of the grid, the (nx/f) x (ny/f) window of
 * every layer around the probe is weighted by A_b exp(-i chi_b) exp(-2 pi i q_b . r_p) / (sqrt(n_beams)
 * sqrt(mx my)) and summed over beams, Fourier transformed, squared (/ (mx my)) and integrated into rings.
 *   s      IN   complex64 [n_beams][ny][nx], DEVICE (page-locked HOST if smatrix_on_host)      beams  IN  HOST [n_beams][2]
 *   out    OUT  fp32 [probes_y][probes_x][n_bins]; device memory or host memory (then copied inside the call)
 *   workspace DEVICE, prism_workspace_bytes(p, PRISM_WS_OUTPUT) */
int prism_compute_output(const prism_params* p, const void* s, const int32_t* beams, int32_t n_beams,
                         float* out, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Conventional multislice (Fig. 1c-e), the comparison path: every probe of the grid
 * is built in Fourier space (hard aperture, exp(-i chi), position phase; sum |psi0|^2 = 1), taken through
 * all slices by the same kernels, and |FFT2(psi_S)|^2 / (nx ny) is integrated into rings.
 *   v, out, workspace as above (workspace: PRISM_WS_MULTISLICE).
 * Square 256- and 512-point grids with a device-resident potential of at most 256 MB of transmission functions run
 * "resident": one launch, one probe per SM in flight from the probe spectrum to the ring sums;
 * `batch` then plays no role.  Results do not depend on the route. */
int multislice_compute_output(const prism_params* p, const float* v, float* out,
                              void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Full diffraction patterns, the paper's "4D output" (PAPER.md:82 "2D, 3D or 4D outputs", :90):
 * the same path as prism_compute_output / multislice_compute_output up to |FFT2|^2, without the ring integration.
 *   patterns OUT DEVICE fp32 [probes_y * probes_x][my][mx] (PRISM: mx = nx / f, my = ny / f, pattern pixel (ky, kx)
 *            at frequency (kx f / lx, ky f / ly); multislice: mx = nx, my = ny), array slot m = signed frequency
 *            index as for the DFT convention above; normalised like the ring output (a pattern sums to at most 1).
 *   Rings of prism_compute_output are sums of these pixels.  workspace: PRISM_WS_OUTPUT / PRISM_WS_MULTISLICE_PATTERNS. */
int prism_compute_patterns(const prism_params* p, const void* s, const int32_t* beams, int32_t n_beams,
                           float* patterns, void* workspace, size_t workspace_bytes, void* cuda_stream);
int multislice_compute_patterns(const prism_params* p, const float* v, float* patterns,
                                void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Arbitrary virtual detectors ("the probe intensity is summed in Fourier space to determine the virtual
 * detector signal"; one detector gives the paper's 2-D output): out[probe][d] = sum over the pattern pixels of
 * masks[d][ky][kx] * I[ky][kx], with the patterns of prism_compute_patterns / multislice_compute_patterns.
 *   masks IN  DEVICE fp32 [n_masks][my][mx] (weights; 0 / 1 for a plain detector), 1 <= n_masks <= 16
 *   out   OUT DEVICE fp32 [probes_y * probes_x][n_masks]
 * Fixed summation order (deterministic).  workspace: PRISM_WS_OUTPUT / PRISM_WS_MULTISLICE_PATTERNS. */
int prism_compute_detectors(const prism_params* p, const void* s, const int32_t* beams, int32_t n_beams,
                            const float* masks, int32_t n_masks, float* out,
                            void* workspace, size_t workspace_bytes, void* cuda_stream);
int multislice_compute_detectors(const prism_params* p, const float* v, const float* masks, int32_t n_masks,
                                 float* out, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Frozen-phonon average ("32 frozen phonon configurations" are averaged): the caller loops over
 * configurations -- each one a full run of the calls above on freshly displaced atoms -- and accumulates
 *   acc[i] = (first ? 0 : acc[i]) + weight * x[i],  i < n      (weight = 1 / n_configurations gives the mean).
 *   acc, x  DEVICE fp32 [n] (any output of the calls above: rings, patterns, detectors). */
int prism_accumulate(float* acc, const float* x, int64_t n, float weight, int32_t first, void* cuda_stream);

/* Text for an error code, and the message of the last CUDA failure seen by the calling thread. */
const char* prism_strerror(int code);
const char* prism_last_error(void);
/* Kernel launches enqueued by this process since the last reset (for launch accounting). */
int64_t prism_launch_count(int32_t reset);

/* Optional device timing per kernel class (measurement aid): when enabled, every
 * launch is bracketed by a pair of CUDA events on the stream it is launched on.  prism_timing_read()
 * waits for the recorded launches, adds their durations (ms) and counts per class into the two arrays
 * (prism_timing_classes() entries each) and clears the record.  The record is process-wide (all threads and
 * streams together, mutex-guarded); off by default.  While it is on, the event between two launches keeps the
 * next kernel's prologue from overlapping the previous kernel, so timed runs are slightly slower. */
int32_t     prism_timing_enable(int32_t enable);          /* returns the previous setting */
int32_t     prism_timing_classes(void);
const char* prism_timing_class_name(int32_t cls);
int         prism_timing_read(double* ms_by_class, int64_t* launches_by_class);

#ifdef __cplusplus
}
#endif
#endif /* PRISM_B200_H */
