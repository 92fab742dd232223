// api.cu -- the C ABI of include/prism.h: parameter checks, fp64 host tables, workspace
// layout and the drivers that enqueue the kernels (B2 "drivers" of SURVEY.md section 1).
//
// Everything that decides an integer (beam membership, band-limit, detector ring of a
// pixel, window origin) is decided here in fp64 and handed to the kernels as tables.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <memory>
#include <mutex>
#include <vector>

#include "../../include/prism.h"
#include "prism_internal.h"

namespace prism {

static thread_local char g_last_error[512] = "";
static std::atomic<long long> g_launches{0};

static int cuda_fail(cudaError_t e, const char* what)
{
    snprintf(g_last_error, sizeof(g_last_error), "%s: %s", what, cudaGetErrorString(e));
    return PRISM_ECUDA;
}
#define CU(call)                                                    \
    do {                                                            \
        cudaError_t e__ = (call);                                   \
        if (e__ != cudaSuccess) return cuda_fail(e__, #call);       \
    } while (0)

// Optional per-kernel-class device timing (prism_timing_enable / prism_timing_read): a pair of
// CUDA events around every launch, on the stream the kernel is launched on.
enum KernelClass { K_POTENTIAL = 0, K_TRANSMISSION, K_ROW_INIT, K_ROW_STEP, K_ROW_FINAL, K_COL_STEP,
                   K_BEAM_SUM, K_BIN_REDUCE, K_COL_MS_INIT, K_COL_MS_FINAL,
                   K_LATTICE_DFT, K_PATTERNS, K_DETECTORS, K_ACCUMULATE, K_WINDOW_OUT, K_MS_RESIDENT, K_NUM_CLASSES };
static const char* const kClassNames[K_NUM_CLASSES] = {
    "potential", "transmission", "row_init", "row_step", "row_final", "col_step", "beam_sum",
    "bin_reduce", "col_ms_init", "col_ms_final", "lattice_dft", "patterns", "detectors", "accumulate", "window_out", "ms_resident" };
struct TimedLaunch { int cls, dev; cudaEvent_t e0, e1; };
// The record is process-wide and guarded by a mutex that is taken only while timing is enabled.  Events belong to the
// device they were created on: the pool of reusable events (creating them costs more than recording) is kept per
// device, and a launch takes its pair from the pool of the device that is current when it is enqueued.
constexpr int TIMING_MAX_DEVICES = 64;
static std::atomic<bool> g_timing{false};
static std::mutex g_timing_mu;
static std::vector<TimedLaunch> g_timed;
static std::vector<cudaEvent_t> g_event_pool[TIMING_MAX_DEVICES];
static cudaError_t take_event_pair(int* dev, cudaEvent_t* e0, cudaEvent_t* e1)
{
    cudaError_t e = cudaGetDevice(dev);
    if (e != cudaSuccess) return e;
    if (*dev < 0 || *dev >= TIMING_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_timing_mu);
    std::vector<cudaEvent_t>& pool = g_event_pool[*dev];
    cudaEvent_t* out[2] = {e0, e1};
    for (int i = 0; i < 2; ++i) {
        if (!pool.empty()) { *out[i] = pool.back(); pool.pop_back(); }
        else if ((e = cudaEventCreate(out[i])) != cudaSuccess) {
            if (i == 1) pool.push_back(*e0);
            return e;
        }
    }
    return cudaSuccess;
}
static void return_event_pair(int dev, cudaEvent_t e0, cudaEvent_t e1)
{
    std::lock_guard<std::mutex> lock(g_timing_mu);
    g_event_pool[dev].push_back(e0);
    g_event_pool[dev].push_back(e1);
}
static void record_timed(int cls, int dev, cudaEvent_t e0, cudaEvent_t e1)
{
    std::lock_guard<std::mutex> lock(g_timing_mu);
    g_timed.push_back({cls, dev, e0, e1});
}

#define LAUNCH(cls, call, stream)                                                      \
    do {                                                                               \
        cudaEvent_t e0__ = nullptr, e1__ = nullptr;                                    \
        int dev__ = 0;                                                                 \
        const bool timed__ = g_timing.load(std::memory_order_relaxed);                 \
        if (timed__) {                                                                 \
            cudaError_t t__ = take_event_pair(&dev__, &e0__, &e1__);                   \
            if (t__ != cudaSuccess) return cuda_fail(t__, "timing events of " #call);  \
            t__ = cudaEventRecord(e0__, (stream));                                     \
            if (t__ != cudaSuccess) { return_event_pair(dev__, e0__, e1__); return cuda_fail(t__, "cudaEventRecord before " #call); } \
        }                                                                              \
        cudaError_t e__ = (call);                                                      \
        if (e__ == cudaSuccess && timed__) e__ = cudaEventRecord(e1__, (stream));      \
        if (e__ != cudaSuccess) {                                                      \
            if (timed__) return_event_pair(dev__, e0__, e1__);                         \
            return cuda_fail(e__, #call);                                              \
        }                                                                              \
        if (timed__) record_timed((cls), dev__, e0__, e1__);                           \
        g_launches.fetch_add(1, std::memory_order_relaxed);                            \
    } while (0)

static const double kPi = 3.14159265358979323846264338327950288;

// ---- physics constants (R0): lambda = h / p, sigma = 2 pi gamma m e lambda / h^2 ----------------
static void electron_constants(double volt, double* lambda_a, double* sigma)
{
    const double h = 6.62607015e-34, c = 299792458.0, e = 1.602176634e-19, m = 9.1093837015e-31;
    const double mc2 = m * c * c, ev = e * volt;
    const double pc = std::sqrt(ev * (ev + 2.0 * mc2));          // momentum * c
    const double lam_m = h * c / pc;
    const double gamma = 1.0 + ev / mc2;
    if (lambda_a) *lambda_a = lam_m * 1e10;
    if (sigma) *sigma = 2.0 * kPi * gamma * m * e * lam_m / (h * h) * 1e-10;
}

static bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }
static int  signed_freq(int slot, int n) { return slot < n / 2 ? slot : slot - n; }

static int check_common(const prism_params* p)
{
    if (!p) return PRISM_EINVAL;
    if (!is_pow2(p->nx) || !is_pow2(p->ny) || p->nx < 64 || p->ny < 64 || p->nx > 2048 || p->ny > 2048) return PRISM_EINVAL;
    if (!(p->cell[0] > 0) || !(p->cell[1] > 0) || !(p->slice_thickness > 0) || p->n_slices < 1) return PRISM_EINVAL;
    if (!(p->voltage > 0)) return PRISM_EINVAL;
    return PRISM_OK;
}
static int check_probe(const prism_params* p)
{
    if (!(p->alpha > 0) || p->probes_x < 1 || p->probes_y < 1) return PRISM_EINVAL;
    if (!(p->det_step > 0) || !(p->det_max > 0) || prism_num_bins(p) < 1 || prism_num_bins(p) > 4096) return PRISM_EINVAL;
    double lambda;
    electron_constants(p->voltage, &lambda, nullptr);
    const double qnyq = std::min(p->nx / (2.0 * p->cell[0]), p->ny / (2.0 * p->cell[1]));
    if (p->alpha / lambda >= 2.0 / 3.0 * qnyq) return PRISM_EINVAL;      // aperture must sit inside the band-limit
    if (p->n_aberrations < 0 || p->n_aberrations > 32 || (p->n_aberrations > 0 && !p->aberrations)) return PRISM_EINVAL;
    for (int i = 0; i < p->n_aberrations; ++i) {
        const prism_aberration& a = p->aberrations[i];
        if (a.n < 1 || a.n > 8 || a.m < 0 || a.m > a.n + 1) return PRISM_EINVAL;
    }
    return PRISM_OK;
}
static int check_prism(const prism_params* p)
{
    if (p->f < 1 || p->nx % p->f || p->ny % p->f) return PRISM_EINVAL;
    const int mx = p->nx / p->f, my = p->ny / p->f;
    if (!is_pow2(mx) || !is_pow2(my)) return PRISM_EINVAL;
    if (mx < 16 || my < 16) return PRISM_EUNSUPPORTED;
    if (mx > 128 || my > 128) return PRISM_EUNSUPPORTED;     // window_out holds 16 .. 128 points per side on chip
    return PRISM_OK;
}

// ---- beams (R4, R7) -----------------------------------------------------------------
static void list_beams(const prism_params* p, std::vector<int32_t>& beams)
{
    double lambda;
    electron_constants(p->voltage, &lambda, nullptr);
    const double qmax = p->alpha / lambda;
    beams.clear();
    for (int ky = -p->ny / 2; ky < p->ny / 2; ++ky) {
        if (ky % p->f) continue;
        for (int kx = -p->nx / 2; kx < p->nx / 2; ++kx) {
            if (kx % p->f) continue;
            const double qx = kx / p->cell[0], qy = ky / p->cell[1];
            if (qx * qx + qy * qy <= qmax * qmax) { beams.push_back(kx); beams.push_back(ky); }
        }
    }
}

// ---- host tables ---------------------------------------------------------------------------------
static void twiddle_table(int n, std::vector<float2>& tw)
{
    tw.resize(n);
    for (int m = 0; m < n; ++m) {
        const double a = -2.0 * kPi * (double)m / (double)n;
        tw[m] = make_float2((float)std::cos(a), (float)std::sin(a));
    }
}

// separable Fresnel propagator (Eq. 2), with an extra real factor folded in
static void propagator_factor(int n, double length, double lambda, double dz, double extra, std::vector<float2>& out)
{
    out.resize(n);
    for (int m = 0; m < n; ++m) {
        const double q = signed_freq(m, n) / length;
        const double a = -kPi * lambda * dz * q * q;
        out[m] = make_float2((float)(extra * std::cos(a)), (float)(extra * std::sin(a)));
    }
}

// 2/3 band-limit (R1): for every kx slot the largest |ky| with q^2 < (2/3 q_nyq)^2, -1 if none
static void band_limit(const prism_params* p, std::vector<int>& ky_lim)
{
    const double qnyq = std::min(p->nx / (2.0 * p->cell[0]), p->ny / (2.0 * p->cell[1]));
    const double qcut2 = (2.0 / 3.0 * qnyq) * (2.0 / 3.0 * qnyq);
    ky_lim.assign(p->nx, -1);
    for (int m = 0; m < p->nx; ++m) {
        const double qx = signed_freq(m, p->nx) / p->cell[0];
        for (int ky = 0; ky <= p->ny / 2; ++ky) {
            const double qy = ky / p->cell[1];
            if (qx * qx + qy * qy < qcut2) ky_lim[m] = ky; else break;
        }
    }
}

// Columns of mixed space that can be non-zero: kx in [0, xband) and [nx - xband, nx), xband a multiple of 32
// (tile widths of the pipelined column pass) that covers every kx with a non-empty band-limited column.
static int band_columns(const prism_params* p)
{
    std::vector<int> lim;
    band_limit(p, lim);
    int kxmax = 0;
    for (int m = 0; m <= p->nx / 2; ++m) if (lim[m] >= 0) kxmax = m;
    return std::min(p->nx / 2, (kxmax + 1 + 31) / 32 * 32);
}
// the same along ky: a multiple of 32 above every ky_lim[kx]
static int band_rows(const prism_params* p)
{
    std::vector<int> lim;
    band_limit(p, lim);
    int kymax = 0;
    for (int m = 0; m < p->nx; ++m) kymax = std::max(kymax, lim[m]);
    return std::min(p->ny / 2, (kymax + 1 + 31) / 32 * 32);
}

// chi(q) (R5, R5b): defocus and spherical aberration, plus the caller's further (n, m) terms
static double aberration(const prism_params* p, double lambda, double qx, double qy)
{
    const double q2 = qx * qx + qy * qy;
    double chi = kPi * lambda * q2 * p->defocus + 0.5 * kPi * p->cs * lambda * lambda * lambda * q2 * q2;
    if (p->n_aberrations > 0) {
        const double theta = lambda * std::sqrt(q2), phi = std::atan2(qy, qx);
        for (int i = 0; i < p->n_aberrations; ++i) {
            const prism_aberration& a = p->aberrations[i];
            chi += 2.0 * kPi / lambda * a.c * std::pow(theta, a.n + 1) / (a.n + 1) * std::cos(a.m * (phi - a.angle));
        }
    }
    return chi;
}

// exp(-2 pi i k pos / length) for every probe coordinate and every listed index k
static void position_phases(int n_probes, double origin, double step, double length,
                            const std::vector<int>& ks, std::vector<float2>& out)
{
    out.resize((size_t)n_probes * ks.size());
    for (int ip = 0; ip < n_probes; ++ip) {
        const double pos = origin + ip * step;
        for (size_t i = 0; i < ks.size(); ++i) {
            double turns = ks[i] * (pos / length);
            turns -= std::floor(turns);
            const double a = -2.0 * kPi * turns;
            out[(size_t)ip * ks.size() + i] = make_float2((float)std::cos(a), (float)std::sin(a));
        }
    }
}

// detector rings (R11): CSR lists of pixel indices per ring for an (my x mx) pattern whose slot
// (ky, kx) is stored TRANSPOSED at kx * my + ky and has frequency (kx fx / lx, ky fy / ly).
static void ring_lists(const prism_params* p, int mx, int my, int fx, int fy,
                       std::vector<int>& start, std::vector<int>& pix)
{
    double lambda;
    electron_constants(p->voltage, &lambda, nullptr);
    const int nb = prism_num_bins(p);
    std::vector<int> bin((size_t)mx * my);
    std::vector<int> count(nb + 1, 0);
    const double ilx2 = 1.0 / (p->cell[0] * p->cell[0]), ily2 = 1.0 / (p->cell[1] * p->cell[1]);
    for (int sx = 0; sx < mx; ++sx) {
        for (int sy = 0; sy < my; ++sy) {
            const double kx = (double)(signed_freq(sx, mx) * fx), ky = (double)(signed_freq(sy, my) * fy);
            const double q = std::sqrt(kx * kx * ilx2 + ky * ky * ily2);
            const double angle = lambda * q;
            const int b = (int)std::floor(angle / p->det_step);
            bin[(size_t)sx * my + sy] = (b < nb) ? b : -1;
            if (b < nb) ++count[b + 1];
        }
    }
    start.assign(nb + 1, 0);
    for (int b = 0; b < nb; ++b) start[b + 1] = start[b] + count[b + 1];
    pix.resize(start[nb]);
    std::vector<int> fill(start.begin(), start.end() - 1);
    for (size_t i = 0; i < bin.size(); ++i)
        if (bin[i] >= 0) pix[fill[bin[i]]++] = (int)i;
}

// ---- workspace bump allocator ----------------------------------------------------------------------
struct Arena {
    char*  base;
    size_t size, used;
    Arena(void* b, size_t s) : base((char*)b), size(s), used(0) {}
    template <class T> T* take(size_t count)
    {
        const size_t bytes = (count * sizeof(T) + 255) / 256 * 256;
        T* ptr = base ? (T*)(base + used) : nullptr;
        used += bytes;
        return ptr;
    }
    bool ok() const { return used <= size; }
};

template <class T>
static cudaError_t upload(T* dst, const std::vector<T>& src, cudaStream_t st)
{
    if (src.empty()) return cudaSuccess;
    return cudaMemcpyAsync(dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice, st);
}

// Host tables are built first and uploaded together afterwards: an upload from pageable memory waits for the work
// already queued on the stream, so interleaving "build a table, upload it" would leave the GPU idle while the
// host builds the next one.  With the uploads deferred, the table building of a call overlaps the kernels the
// previous call left running.
struct DeferredUploads {
    struct Item { void* dst; const void* src; size_t bytes; std::shared_ptr<void> keep; };
    std::vector<Item> items;
    template <class T> void add(T* dst, std::vector<T>&& src)
    {
        if (src.empty()) return;
        auto keep = std::make_shared<std::vector<T>>(std::move(src));
        items.push_back({dst, keep->data(), keep->size() * sizeof(T), keep});
    }
    template <class T> void add(T* dst, const std::vector<T>& src) { add(dst, std::vector<T>(src)); }
    cudaError_t flush(cudaStream_t st)
    {
        for (const Item& it : items) {
            cudaError_t e = cudaMemcpyAsync(it.dst, it.src, it.bytes, cudaMemcpyHostToDevice, st);
            if (e != cudaSuccess) return e;
        }
        return cudaSuccess;
    }
};

static int default_probe_batch(const prism_params* p, size_t bytes_per_probe)
{
    long long n = (long long)p->probes_x * p->probes_y;
    // default: about 4 GiB of waves per batch (enough to hide a streamed potential behind the passes)
    long long b = p->batch > 0 ? p->batch : std::max<long long>(1, (long long)(4ull << 30) / (long long)bytes_per_probe);
    return (int)std::min(n, b);
}

// ---- potential slices: resident, or streamed from page-locked host memory -------
// A ring of RING raw slices is filled over a private copy stream; the (tiny) transmission kernel
// turns the slice into t_s = exp(i sigma V_s) on the main stream and frees the ring slot.
struct SliceFeeder {
    static constexpr int RING = 3;
    const float* v = nullptr;
    bool on_host = false;
    int64_t npix = 0;
    int n_slices = 0;
    double sigma = 0;
    bool pairs = false;                 // transmission function in pair layout (packed row pass)
    float2* tbuf = nullptr;             // t_s of the current slice; or of every slice when t_slices == n_slices
    int t_slices = 1;                   // slices of t kept (small stacks keep all of them across wave batches)
    int t_done = 0;                     // slices [0, t_done) of a kept stack are already computed
    float2* current = nullptr;          // t_s the next passes read
    float* ring[RING] = {nullptr, nullptr, nullptr};
    cudaStream_t main_stream = nullptr, copy_stream = nullptr;
    cudaEvent_t filled[RING] = {}, consumed[RING] = {};
    bool slot_used[RING] = {false, false, false};
    int next_copy = 0;

    int init()
    {
        if (!on_host) return PRISM_OK;
        CU(cudaStreamCreateWithFlags(&copy_stream, cudaStreamNonBlocking));
        for (int r = 0; r < RING; ++r) {
            CU(cudaEventCreateWithFlags(&filled[r], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&consumed[r], cudaEventDisableTiming));
        }
        // copies must not start before earlier work on the main stream that may still use the ring
        cudaEvent_t start;
        CU(cudaEventCreateWithFlags(&start, cudaEventDisableTiming));
        CU(cudaEventRecord(start, main_stream));
        CU(cudaStreamWaitEvent(copy_stream, start, 0));
        CU(cudaEventDestroy(start));
        return PRISM_OK;
    }
    void begin_sweep() { next_copy = 0; }
    int prefetch(int upto)
    {
        for (; next_copy < std::min(n_slices, upto); ++next_copy) {
            const int r = next_copy % RING;
            if (slot_used[r]) CU(cudaStreamWaitEvent(copy_stream, consumed[r], 0));
            CU(cudaMemcpyAsync(ring[r], v + (size_t)next_copy * npix, npix * sizeof(float),
                               cudaMemcpyHostToDevice, copy_stream));
            CU(cudaEventRecord(filled[r], copy_stream));
            slot_used[r] = true;
        }
        return PRISM_OK;
    }
    // enqueue everything needed so that tbuf holds t_s for the kernels enqueued next on main_stream
    int get(int s)
    {
        const float* src = v + (size_t)s * npix;
        if (on_host) {
            int rc = prefetch(s + RING);
            if (rc) return rc;
            const int r = s % RING;
            CU(cudaStreamWaitEvent(main_stream, filled[r], 0));
            src = ring[r];
        }
        if (t_slices > 1) {
            current = tbuf + (size_t)s * npix;
            if (s < t_done) return PRISM_OK;        // computed by an earlier wave batch
            t_done = s + 1;
        } else {
            current = tbuf;
        }
        LAUNCH(K_TRANSMISSION, launch_transmission(src, current, sigma, npix, pairs, main_stream), main_stream);
        if (on_host) CU(cudaEventRecord(consumed[s % RING], main_stream));
        return PRISM_OK;
    }
    void release()
    {
        if (!on_host) return;
        for (int r = 0; r < RING; ++r) {
            if (filled[r]) cudaEventDestroy(filled[r]);
            if (consumed[r]) cudaEventDestroy(consumed[r]);
        }
        if (copy_stream) cudaStreamDestroy(copy_stream);
    }
};

// tables every slice loop needs
struct SliceTables {
    float2 *tw_x, *tw_y, *prop_x, *prop_y;
    int* ky_lim;
};
static void carve_slice_tables(Arena& a, const prism_params* p, SliceTables& t)
{
    t.tw_x = a.take<float2>(p->nx);
    t.tw_y = a.take<float2>(p->ny);
    t.prop_x = a.take<float2>(p->nx);
    t.prop_y = a.take<float2>(p->ny);
    t.ky_lim = a.take<int>(p->nx);
}
static void fill_slice_tables(const prism_params* p, const SliceTables& t, DeferredUploads& up)
{
    double lambda;
    electron_constants(p->voltage, &lambda, nullptr);
    std::vector<float2> h;
    twiddle_table(p->nx, h);
    up.add(t.tw_x, std::move(h));
    twiddle_table(p->ny, h);
    up.add(t.tw_y, std::move(h));
    // the row pass runs unscaled inverse FFTs and so does the column pass: fold 1/nx and 1/ny here
    propagator_factor(p->nx, p->cell[0], lambda, p->slice_thickness, 1.0 / p->nx, h);
    up.add(t.prop_x, std::move(h));
    propagator_factor(p->ny, p->cell[1], lambda, p->slice_thickness, 1.0 / p->ny, h);
    up.add(t.prop_y, std::move(h));
    std::vector<int> lim;
    band_limit(p, lim);
    up.add(t.ky_lim, std::move(lim));
}
static void carve_feeder(Arena& a, const prism_params* p, SliceFeeder& f, bool many_batches)
{
    const size_t npix = (size_t)p->nx * p->ny;
    // a resident potential whose transmission functions fit in 256 MiB keeps all of them, so that later wave
    // batches (multislice probes) do not recompute them
    f.t_slices = (many_batches && !p->potential_on_host && (size_t)p->n_slices * npix * sizeof(float2) <= ((size_t)256 << 20)) ? p->n_slices : 1;
    f.tbuf = a.take<float2>(npix * f.t_slices);
    if (p->potential_on_host)
        for (int r = 0; r < SliceFeeder::RING; ++r) f.ring[r] = a.take<float>(npix);
}

// ---- layouts -----------------------------------------------------------------------------------------
// beams per batch of prism_compute_smatrix: all of them when S is device memory (it is the wave buffer); with S in
// host memory the batch lives in the workspace: p->batch beams, by default about 4 GiB of waves (two such buffers
// alternate, so that the copy-out of one batch overlaps the propagation of the next)
static int smatrix_batch(const prism_params* p, int n_beams)
{
    if (p->batch > 0) return std::min<int>(p->batch, n_beams);
    if (!p->smatrix_on_host) return n_beams;
    // at least four batches, so that the copy-out of one overlaps the propagation of the next
    const long long per_beam = (long long)p->nx * p->ny * (long long)sizeof(float2);
    const long long by_mem = std::max<long long>(1, (long long)(4ull << 30) / per_beam);
    return (int)std::max<long long>(1, std::min<long long>(by_mem, (n_beams + 3) / 4));
}
// Grids on the blocked mixed-space layout (blocked_grid): the last row pass turns blocked mixed space into natural
// real space, which cannot be done in place, so it runs FINAL_CHUNK waves at a time into a staging buffer that is
// then copied over the waves' own storage (or straight to a host S-matrix, from two alternating staging buffers).
constexpr int FINAL_CHUNK = 16;
struct SmatrixLayout {
    SliceTables tab; SliceFeeder feed; int2* beams;
    float2* wave; int wave_bufs;                 // S in host memory: wave_bufs batches of waves
    float2* final_stage; int final_chunk, final_bufs;
};
static void layout_smatrix(Arena& a, const prism_params* p, int n_beams, SmatrixLayout& L)
{
    const bool blocked = blocked_grid(p->nx, p->ny), on_host = p->smatrix_on_host != 0;
    const int batch = smatrix_batch(p, n_beams);
    carve_slice_tables(a, p, L.tab);
    carve_feeder(a, p, L.feed, on_host && batch < n_beams);
    L.beams = a.take<int2>(n_beams);
    L.wave_bufs = !on_host ? 0 : (blocked || batch >= n_beams) ? 1 : 2;
    L.wave = on_host ? a.take<float2>((size_t)L.wave_bufs * batch * p->nx * p->ny) : nullptr;
    L.final_chunk = blocked ? std::min(FINAL_CHUNK, std::max(1, n_beams)) : 0;
    L.final_bufs = !blocked ? 0 : on_host ? 2 : 1;
    L.final_stage = blocked ? a.take<float2>((size_t)L.final_bufs * L.final_chunk * p->nx * p->ny) : nullptr;
}

constexpr int LATTICE_MAX_SLOTS = 4, LATTICE_MAX_Q = 32;
struct OutputLayout {
    float2 *tw_x, *tw_y, *coef_b, *phase_x, *phase_y, *w, *lat_coef, *slab;
    int slab_rows;
    int *win_x0, *win_y0, *bin_start, *bin_pix, *cell_beam;
    float *intensity, *out_stage;
    int batch;
};
static void layout_output(Arena& a, const prism_params* p, int n_beams, OutputLayout& L)
{
    const int mx = p->nx / p->f, my = p->ny / p->f, nb = prism_num_bins(p);
    const size_t npix = (size_t)mx * my;
    L.batch = default_probe_batch(p, npix * 12);
    L.slab = nullptr; L.slab_rows = 0;
    if (p->smatrix_on_host) {
        // S in host memory: a batch is whole probe rows, and the workspace holds a ring of the pixel rows of every layer
        // that the current and the next batch's windows cover (at most ~16 GiB: fewer probe rows per batch otherwise),
        // so the copies of batch k + 1 run while batch k computes and every row is copied once per sweep
        const int sy = std::max(1, (int)std::floor(p->probe_step[1] / (p->cell[1] / p->ny) + 0.5));
        int rows = std::min(p->probes_y, std::max(1, L.batch / std::max(1, p->probes_x)));
        auto ring_rows = [&](int r) {
            const int pix = std::min(p->ny, sy * (r - 1) + my);                   // rows of one batch
            return r >= p->probes_y ? pix : pix + std::min(pix, sy * r);         // + the rows the next batch adds
        };
        while (rows > 1 && (size_t)n_beams * ring_rows(rows) * p->nx * sizeof(float2) > ((size_t)16 << 30)) rows /= 2;
        L.batch = rows * p->probes_x;
        L.slab_rows = ring_rows(rows);
    }
    L.tw_x = a.take<float2>(mx);
    L.tw_y = a.take<float2>(my);
    L.coef_b = a.take<float2>(n_beams);
    L.phase_x = a.take<float2>((size_t)p->probes_x * n_beams);
    L.phase_y = a.take<float2>((size_t)p->probes_y * n_beams);
    L.win_x0 = a.take<int>(p->probes_x);
    L.win_y0 = a.take<int>(p->probes_y);
    L.bin_start = a.take<int>(nb + 1);
    L.bin_pix = a.take<int>(npix);
    L.lat_coef = a.take<float2>(n_beams);
    L.cell_beam = a.take<int>((size_t)LATTICE_MAX_SLOTS * LATTICE_MAX_Q * LATTICE_MAX_Q);
    L.w = a.take<float2>((size_t)L.batch * npix);
    L.intensity = a.take<float>((size_t)L.batch * npix);
    L.out_stage = a.take<float>((size_t)p->probes_x * p->probes_y * nb);
    if (p->smatrix_on_host) L.slab = a.take<float2>((size_t)n_beams * L.slab_rows * p->nx);
}

// Regular probe lattice test ("lattice DFT"): the window origins advance by a constant
// power-of-two number of pixels s that divides the window, the probe step is exactly s pixels, and every
// beam index is a multiple of f.  Decided on the integer origin tables and in fp64.
struct LatticePlan {
    bool ok = false;
    int q = 0, sx_log2 = 0, sy_log2 = 0, n_slots = 0;
    std::vector<int> cell_beam;
};
static int regular_step(const std::vector<int>& w0, int n, int m, double step_px)
{
    if (w0.size() < 2) return 0;
    const int s = ((w0[1] - w0[0]) % n + n) % n;
    if (s < 1 || !is_pow2(s) || m % s) return 0;
    for (size_t i = 1; i < w0.size(); ++i)
        if ((((w0[i] - w0[i - 1]) % n) + n) % n != s) return 0;
    if (std::fabs(step_px - (double)s) > 1e-9) return 0;
    if ((long long)w0.size() * s > n) return 0;                   // every probe owns a distinct lattice site
    return s;
}
static LatticePlan plan_lattice(const prism_params* p, const int32_t* beams, int n_beams,
                                const std::vector<int>& wx0, const std::vector<int>& wy0, int mx, int my)
{
    LatticePlan L;
    const int sx = regular_step(wx0, p->nx, mx, p->probe_step[0] / (p->cell[0] / p->nx));
    const int sy = regular_step(wy0, p->ny, my, p->probe_step[1] / (p->cell[1] / p->ny));
    if (!sx || !sy || mx / sx != my / sy) return L;
    const int q = mx / sx;
    if (q != 8 && q != 16 && q != 32) return L;
    std::vector<int> count((size_t)q * q, 0);
    L.cell_beam.assign((size_t)LATTICE_MAX_SLOTS * q * q, -1);
    for (int b = 0; b < n_beams; ++b) {
        const int kx = beams[2 * b], ky = beams[2 * b + 1];
        if (kx % p->f || ky % p->f) return L;
        const int m = ((kx / p->f) % q + q) % q, n = ((ky / p->f) % q + q) % q;
        const int c = n * q + m;
        if (count[c] >= LATTICE_MAX_SLOTS) return L;
        L.cell_beam[(size_t)count[c] * q * q + c] = b;
        L.n_slots = std::max(L.n_slots, ++count[c]);
    }
    for (L.sx_log2 = 0; (1 << L.sx_log2) < sx; ++L.sx_log2) {}
    for (L.sy_log2 = 0; (1 << L.sy_log2) < sy; ++L.sy_log2) {}
    L.q = q;
    L.ok = L.n_slots >= 1;
    return L;
}

// ---- S-matrix in host memory, stage 2 ("the current S-matrix subset") -----------------------------
// The device holds a ring of pixel rows of every layer.  Rows are numbered by the unwrapped offset u from the first
// window row of probe row 0 (pixel row (y00 + u) mod ny); probe-row batch k needs u in [sy R k, sy R k + pix_k) and
// row u sits at ring row u % cap.  Each batch copies only the rows the ring does not hold yet, on a private copy
// stream: with cap >= rows of a batch + rows the next batch adds, the copies of batch k + 1 overlap the kernels of
// batch k (they wait for batch k - 1, whose rows they overwrite).  That holds whenever consecutive batches share or
// abut pixel rows (probe-row step <= window side, every lattice the configs use).  When they leave a gap
// (sy * rows_per_batch > rows of a batch) the ring is 2 x a batch deep but row u % cap of batch k + 1 can land on rows
// batch k still reads, so copy_batch(k + 1) waits for done[k]: correct, not overlapped.
struct SlabRing {
    const char* s = nullptr;            // host S-matrix [n_beams][ny][nx] complex64
    char* slab = nullptr;               // device ring [n_beams][cap][nx]
    int cap = 0, n_beams = 0, nx = 0, ny = 0, my = 0, sy = 1, y00 = 0, rows_per_batch = 1, probes_y = 0;
    long long have_hi = -1;             // rows [.., have_hi) of the newest batch are in the ring or on their way
    cudaStream_t main_stream = nullptr, copy_stream = nullptr;
    std::vector<cudaEvent_t> copied, done;

    int n_batches() const { return (probes_y + rows_per_batch - 1) / rows_per_batch; }
    int u_first(int k) const { return sy * rows_per_batch * k; }
    int pix_rows(int k) const
    {
        const int r = std::min(rows_per_batch, probes_y - k * rows_per_batch);
        return std::min(ny, sy * (r - 1) + my);
    }
    int init()
    {
        CU(cudaStreamCreateWithFlags(&copy_stream, cudaStreamNonBlocking));
        copied.assign(n_batches(), nullptr);
        done.assign(n_batches(), nullptr);
        for (int k = 0; k < n_batches(); ++k) {
            CU(cudaEventCreateWithFlags(&copied[k], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&done[k], cudaEventDisableTiming));
        }
        // the ring may still be in use by earlier work on the main stream
        cudaEvent_t start;
        CU(cudaEventCreateWithFlags(&start, cudaEventDisableTiming));
        CU(cudaEventRecord(start, main_stream));
        CU(cudaStreamWaitEvent(copy_stream, start, 0));
        CU(cudaEventDestroy(start));
        return PRISM_OK;
    }
    // enqueue the copies batch k still needs; called in batch order, batch k + 1 right after batch k's kernel
    int copy_batch(int k)
    {
        const long long a = u_first(k), b = a + pix_rows(k);
        if (b - a > cap) return PRISM_ENOMEM;
        long long c0 = std::max(a, have_hi < 0 ? a : have_hi);
        // rows [c0 - cap, b - cap) are overwritten: wait for the newest earlier batch that still reads any of them
        for (int j = k - 1; j >= 0; --j)
            if (b - cap > u_first(j)) { CU(cudaStreamWaitEvent(copy_stream, done[j], 0)); break; }
        const size_t row_bytes = (size_t)nx * sizeof(float2);
        for (long long u = c0; u < b;) {
            const int slot = (int)(u % cap), y = (int)((y00 + u) % ny);
            const long long seg = std::min<long long>(std::min<long long>(b - u, cap - slot), ny - y);
            CU(cudaMemcpy2DAsync(slab + (size_t)slot * row_bytes, (size_t)cap * row_bytes,
                                 s + (size_t)y * row_bytes, (size_t)ny * row_bytes,
                                 (size_t)seg * row_bytes, n_beams, cudaMemcpyHostToDevice, copy_stream));
            u += seg;
        }
        have_hi = b;
        CU(cudaEventRecord(copied[k], copy_stream));
        return PRISM_OK;
    }
    void release()
    {
        for (cudaEvent_t e : copied) if (e) cudaEventDestroy(e);
        for (cudaEvent_t e : done) if (e) cudaEventDestroy(e);
        copied.clear(); done.clear();
        if (copy_stream) { cudaStreamDestroy(copy_stream); copy_stream = nullptr; }
    }
};

struct MultisliceLayout {
    SliceTables tab;
    SliceFeeder feed;
    float2 *aperture_t, *phase_x, *phase_y, *psi;
    int *bin_start, *bin_pix;
    float *intensity, *out_stage;
    int batch, waves;
};
// plain multislice runs resident (ms_resident.cu: one probe per SM, one launch for all slices) when the grid is one
// of its sizes and the transmission functions of all slices are kept in device memory
static bool multislice_resident(const prism_params* p)
{
    return resident_grid(p->nx, p->ny) && !p->potential_on_host &&
           (size_t)p->n_slices * p->nx * p->ny * sizeof(float2) <= ((size_t)256 << 20);
}
// `rings`: the call integrates into rings and so may take the resident route; patterns and mask detectors always
// run per pass and need a batch of waves only.  RESIDENT_SLOTS is a cap on the waves in flight (the launch takes
// min(probes, slots, SMs of the device)), kept a constant so that prism_workspace_bytes stays host-only.
static void layout_multislice(Arena& a, const prism_params* p, MultisliceLayout& L, bool rings)
{
    const size_t npix = (size_t)p->nx * p->ny;
    const int nb = prism_num_bins(p);
    L.batch = default_probe_batch(p, npix * 12);
    // wave slots: a batch of the per-pass path, or one per SM for the resident kernel
    L.waves = L.batch;
    if (rings && multislice_resident(p))
        L.waves = std::max<long long>(L.batch, std::min<long long>((long long)p->probes_x * p->probes_y, RESIDENT_SLOTS));
    carve_slice_tables(a, p, L.tab);
    carve_feeder(a, p, L.feed, true);
    L.aperture_t = a.take<float2>(npix);
    L.phase_x = a.take<float2>((size_t)p->probes_x * p->nx);
    L.phase_y = a.take<float2>((size_t)p->probes_y * p->ny);
    L.bin_start = a.take<int>(nb + 1);
    L.bin_pix = a.take<int>(npix);
    L.psi = a.take<float2>((size_t)L.waves * npix);
    L.intensity = a.take<float>((size_t)L.waves * npix);
    L.out_stage = a.take<float>((size_t)p->probes_x * p->probes_y * nb);
}

constexpr int POT_TILE = 16;
constexpr int POT_CHUNK_SLICES = 8;
struct PotentialLayout { int* cell_start; float* lut_v; double* lut_rcut; float* stage; };
static void layout_potential(Arena& a, const prism_params* p, int n_luts, int lut_n, PotentialLayout& L)
{
    const size_t cells = (size_t)p->n_slices * (p->nx / POT_TILE) * (p->ny / POT_TILE);
    L.cell_start = a.take<int>(cells + 1);
    L.lut_v = a.take<float>((size_t)std::max(1, n_luts) * std::max(2, lut_n));
    L.lut_rcut = a.take<double>(std::max(1, n_luts));
    L.stage = p->potential_on_host ? a.take<float>((size_t)2 * POT_CHUNK_SLICES * p->nx * p->ny) : nullptr;   // two alternating chunks
}

// Results that leave for page-locked host memory while the next piece is computed: two alternating device buffers and
// a private copy stream.  acquire(i): the main stream may overwrite buffer i; send(i, ...): buffer i has just been
// filled on the main stream and is copied out; join(): the main stream waits for everything sent.
struct HostCopyOut {
    cudaStream_t stream = nullptr;
    cudaEvent_t ready[2] = {nullptr, nullptr}, freed[2] = {nullptr, nullptr};
    bool used[2] = {false, false};
    int init()
    {
        CU(cudaStreamCreateWithFlags(&stream, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            CU(cudaEventCreateWithFlags(&ready[i], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&freed[i], cudaEventDisableTiming));
        }
        return PRISM_OK;
    }
    int acquire(int i, cudaStream_t st)
    {
        if (used[i]) CU(cudaStreamWaitEvent(st, freed[i], 0));
        return PRISM_OK;
    }
    int send(int i, void* dst, const void* src, size_t bytes, cudaStream_t st)
    {
        CU(cudaEventRecord(ready[i], st));
        CU(cudaStreamWaitEvent(stream, ready[i], 0));
        CU(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, stream));
        CU(cudaEventRecord(freed[i], stream));
        used[i] = true;
        return PRISM_OK;
    }
    int join(cudaStream_t st)
    {
        for (int i = 0; i < 2; ++i)
            if (used[i]) CU(cudaStreamWaitEvent(st, freed[i], 0));
        return PRISM_OK;
    }
    ~HostCopyOut()
    {
        for (int i = 0; i < 2; ++i) { if (ready[i]) cudaEventDestroy(ready[i]); if (freed[i]) cudaEventDestroy(freed[i]); }
        if (stream) cudaStreamDestroy(stream);
    }
};

static bool pointer_is_device(const void* ptr)
{
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, ptr) != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

}  // namespace prism

using namespace prism;

// =========================================================================================================
extern "C" {
#pragma GCC visibility push(default)

const char* prism_strerror(int code)
{
    switch (code) {
        case PRISM_OK: return "ok";
        case PRISM_EINVAL: return "invalid argument";
        case PRISM_ENOMEM: return "workspace too small";
        case PRISM_ECUDA: return "CUDA error";
        case PRISM_EUNSUPPORTED: return "unsupported configuration";
        case PRISM_ENOLUT: return "no lookup table for an atom's Z";
    }
    return "unknown error";
}
const char* prism_last_error(void) { return g_last_error; }

int64_t prism_launch_count(int32_t reset)
{
    return reset ? g_launches.exchange(0) : g_launches.load();
}

int32_t prism_timing_enable(int32_t enable)
{
    return g_timing.exchange(enable != 0) ? 1 : 0;
}

int32_t prism_timing_classes(void) { return K_NUM_CLASSES; }
const char* prism_timing_class_name(int32_t cls) { return (cls >= 0 && cls < K_NUM_CLASSES) ? kClassNames[cls] : ""; }

int prism_timing_read(double* ms_by_class, int64_t* launches_by_class)
{
    if (!ms_by_class || !launches_by_class) return PRISM_EINVAL;
    for (int c = 0; c < K_NUM_CLASSES; ++c) { ms_by_class[c] = 0.0; launches_by_class[c] = 0; }
    std::lock_guard<std::mutex> lock(g_timing_mu);
    // every entry leaves the record as it is read and its events go back to their device's pool exactly once, also
    // when a CUDA call fails part-way: the entries not yet read stay for the next call
    while (!g_timed.empty()) {
        const TimedLaunch t = g_timed.back();
        g_timed.pop_back();
        float ms = 0.f;
        cudaError_t e = cudaEventSynchronize(t.e1);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, t.e0, t.e1);
        g_event_pool[t.dev].push_back(t.e0);
        g_event_pool[t.dev].push_back(t.e1);
        if (e != cudaSuccess) return cuda_fail(e, "prism_timing_read");
        ms_by_class[t.cls] += ms;
        ++launches_by_class[t.cls];
    }
    return PRISM_OK;
}

int prism_accumulate(float* acc, const float* x, int64_t n, float weight, int32_t first, void* cuda_stream)
{
    if (!acc || !x || n < 0) return PRISM_EINVAL;
    if (!pointer_is_device(acc) || !pointer_is_device(x)) return PRISM_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    LAUNCH(K_ACCUMULATE, launch_accumulate(acc, x, n, weight, first != 0, st), st);
    return PRISM_OK;
}

int prism_constants(double voltage, double* lambda, double* sigma)
{
    if (!(voltage > 0)) return PRISM_EINVAL;
    electron_constants(voltage, lambda, sigma);
    return PRISM_OK;
}

int32_t prism_num_bins(const prism_params* p)
{
    if (!p || !(p->det_step > 0)) return 0;
    return (int32_t)std::floor(p->det_max / p->det_step + 0.5);
}

int32_t prism_band_columns(const prism_params* p)
{
    if (check_common(p)) return 0;
    return band_columns(p);
}

int prism_num_beams(const prism_params* p, int32_t* n_beams)
{
    if (!n_beams) return PRISM_EINVAL;
    int rc = check_common(p);
    if (rc) return rc;
    if ((rc = check_probe(p))) return rc;
    if (p->f < 1 || p->nx % p->f || p->ny % p->f) return PRISM_EINVAL;
    std::vector<int32_t> beams;
    list_beams(p, beams);
    *n_beams = (int32_t)(beams.size() / 2);
    return PRISM_OK;
}

size_t prism_workspace_bytes(const prism_params* p, int32_t which)
{
    if (check_common(p)) return 0;
    Arena a(nullptr, 0);
    switch (which) {
        case PRISM_WS_SMATRIX: {
            int32_t nb = 0;
            if (prism_num_beams(p, &nb)) return 0;
            SmatrixLayout L;
            layout_smatrix(a, p, nb, L);
            break;
        }
        case PRISM_WS_OUTPUT: {
            int32_t nb = 0;
            if (prism_num_beams(p, &nb) || check_prism(p)) return 0;
            OutputLayout L;
            layout_output(a, p, nb, L);
            break;
        }
        case PRISM_WS_MULTISLICE: {
            if (check_probe(p)) return 0;
            MultisliceLayout L;
            layout_multislice(a, p, L, true);
            break;
        }
        case PRISM_WS_MULTISLICE_PATTERNS: {
            if (check_probe(p)) return 0;
            MultisliceLayout L;
            layout_multislice(a, p, L, false);
            break;
        }
        case PRISM_WS_POTENTIAL: {
            PotentialLayout L;
            layout_potential(a, p, 128, 4096, L);       // room for 128 species x 4096 samples; atoms are extra
            break;
        }
        default: return 0;
    }
    return a.used + 256;
}

// ---------------------------------------------------------------------------------------------------------
int prism_build_potential(const prism_params* p, const double* atoms_xyz, const int32_t* z_number,
                          int64_t n_atoms, const prism_lut* luts, int32_t n_luts, float* v,
                          void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    int rc = check_common(p);
    if (rc) return rc;
    if (n_atoms < 0 || (n_atoms > 0 && (!atoms_xyz || !z_number)) || !v || !workspace) return PRISM_EINVAL;
    if (n_luts < 0 || n_luts > 128 || (n_atoms > 0 && (n_luts == 0 || !luts))) return PRISM_EINVAL;
    if (n_atoms > (int64_t)0x7fffffff) return PRISM_EUNSUPPORTED;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int lut_n = 2;
    double rc_max = 0.0;
    for (int l = 0; l < n_luts; ++l) {
        if (!luts[l].v || luts[l].n < 2 || luts[l].n > 4096 || !(luts[l].r_cut > 0)) return PRISM_EINVAL;
        if (l > 0 && luts[l].n != luts[0].n) return PRISM_EUNSUPPORTED;       // one table length per call
        lut_n = luts[l].n;
        rc_max = std::max(rc_max, luts[l].r_cut);
    }
    if (2.0 * rc_max >= p->cell[0] || 2.0 * rc_max >= p->cell[1]) return PRISM_EINVAL;

    const int nx = p->nx, ny = p->ny, ns = p->n_slices;
    const int tiles_x = nx / POT_TILE, tiles_y = ny / POT_TILE;
    const double px = p->cell[0] / nx, py = p->cell[1] / ny;
    const size_t cells = (size_t)ns * tiles_x * tiles_y;

    Arena a(workspace, workspace_bytes);
    PotentialLayout L;
    layout_potential(a, p, 128, 4096, L);
    PotAtom* d_atoms = a.take<PotAtom>((size_t)n_atoms);
    if (!a.ok()) return PRISM_ENOMEM;

    // host: slice + tile of every atom, counting sort by cell (stable: original order inside a cell)
    std::vector<int> cell_of((size_t)n_atoms);
    std::vector<int> start(cells + 1, 0);
    std::vector<PotAtom> sorted((size_t)n_atoms);
    std::vector<PotAtom> tmp((size_t)n_atoms);
    for (int64_t i = 0; i < n_atoms; ++i) {
        int lut = -1;
        for (int l = 0; l < n_luts; ++l) if (luts[l].z == z_number[i]) lut = l;
        if (lut < 0) return PRISM_ENOLUT;
        double x = atoms_xyz[3 * i], y = atoms_xyz[3 * i + 1], z = atoms_xyz[3 * i + 2];
        x -= p->cell[0] * std::floor(x / p->cell[0]);
        y -= p->cell[1] * std::floor(y / p->cell[1]);
        int s = (int)std::floor(z / p->slice_thickness);
        s = std::min(std::max(s, 0), ns - 1);
        int ix = std::min(std::max((int)std::floor(x / px), 0), nx - 1);
        int iy = std::min(std::max((int)std::floor(y / py), 0), ny - 1);
        const int cell = (s * tiles_y + iy / POT_TILE) * tiles_x + ix / POT_TILE;
        cell_of[i] = cell;
        ++start[cell + 1];
        tmp[i].x = x; tmp[i].y = y; tmp[i].lut = lut; tmp[i].pad = 0;
    }
    for (size_t c = 0; c < cells; ++c) start[c + 1] += start[c];
    {
        std::vector<int> fill(start.begin(), start.end() - 1);
        for (int64_t i = 0; i < n_atoms; ++i) sorted[fill[cell_of[i]]++] = tmp[i];
    }
    std::vector<float> h_lut((size_t)std::max(1, n_luts) * lut_n, 0.f);
    std::vector<double> h_rcut(std::max(1, n_luts), 1.0);
    for (int l = 0; l < n_luts; ++l) {
        std::memcpy(&h_lut[(size_t)l * lut_n], luts[l].v, sizeof(float) * lut_n);
        h_rcut[l] = luts[l].r_cut;
    }
    CU(upload(L.cell_start, start, st));
    CU(upload(L.lut_v, h_lut, st));
    CU(upload(L.lut_rcut, h_rcut, st));
    CU(upload(d_atoms, sorted, st));
    CU(cudaStreamSynchronize(st));          // the sorted host vectors are local; the kernels below run asynchronously

    PotentialArgs g;
    g.atoms = d_atoms; g.cell_start = L.cell_start; g.lut_v = L.lut_v; g.lut_rcut = L.lut_rcut; g.lut_n = lut_n;
    g.nx = nx; g.ny = ny; g.tiles_x = tiles_x; g.tiles_y = tiles_y; g.tile = POT_TILE;
    const double reach_px = std::max(rc_max / px, rc_max / py);
    g.reach_tiles = (int)std::ceil(reach_px / POT_TILE);
    g.px = px; g.py = py; g.lx = p->cell[0]; g.ly = p->cell[1];
    const size_t npix = (size_t)nx * ny;
    if (!p->potential_on_host) {
        // grid.y is limited to 65535 slices per launch
        for (int s0 = 0; s0 < ns; s0 += 32768) {
            g.slice0 = s0; g.n_slices_chunk = std::min(32768, ns - s0); g.v_out = v + (size_t)s0 * npix;
            LAUNCH(K_POTENTIAL, launch_potential(g, st), st);
        }
    } else {
        // chunks of slices are built in one of two staging buffers and leave over a private copy stream while the
        // next chunk is built
        HostCopyOut out;
        if ((rc = out.init())) return rc;
        int n_chunk = 0;
        for (int s0 = 0; s0 < ns; s0 += POT_CHUNK_SLICES, ++n_chunk) {
            const int b = n_chunk % 2;
            float* stage = L.stage + (size_t)b * POT_CHUNK_SLICES * npix;
            g.slice0 = s0; g.n_slices_chunk = std::min(POT_CHUNK_SLICES, ns - s0); g.v_out = stage;
            if ((rc = out.acquire(b, st))) return rc;
            LAUNCH(K_POTENTIAL, launch_potential(g, st), st);
            if ((rc = out.send(b, v + (size_t)s0 * npix, stage, (size_t)g.n_slices_chunk * npix * sizeof(float), st))) return rc;
        }
        if ((rc = out.join(st))) return rc;
    }
    return PRISM_OK;
}

// ---------------------------------------------------------------------------------------------------------
// The same call on the library's built-in scratch array (potential.cu) instead of a caller workspace: for callers
// that may not allocate device memory.  Nothing here allocates on the device; the size is checked first so that an
// oversized request fails with the numbers in prism_last_error() instead of a bare PRISM_ENOMEM.
static_assert(PRISM_STATIC_SCRATCH_BYTES == POT_STATIC_BYTES, "prism.h and potential.cu disagree on the scratch size");
int prism_build_potential_static(const prism_params* p, const double* atoms_xyz, const int32_t* z_number,
                                 int64_t n_atoms, const prism_lut* luts, int32_t n_luts, float* v,
                                 void* cuda_stream)
{
    int rc = check_common(p);
    if (rc) return rc;
    if (n_atoms < 0) return PRISM_EINVAL;
    if (p->potential_on_host) {
        snprintf(g_last_error, sizeof(g_last_error),
                 "prism_build_potential_static: potential_on_host needs staging buffers and a copy stream; v must be device memory");
        return PRISM_EUNSUPPORTED;
    }
    const size_t fixed = prism_workspace_bytes(p, PRISM_WS_POTENTIAL);
    const size_t atoms = (size_t)std::min<int64_t>(n_atoms, (int64_t)PRISM_STATIC_SCRATCH_BYTES);     // beyond that it cannot fit anyway
    const size_t need = fixed + 512 + atoms * sizeof(PotAtom);
    if (fixed == 0 || need > PRISM_STATIC_SCRATCH_BYTES) {
        snprintf(g_last_error, sizeof(g_last_error),
                 "prism_build_potential_static: %zu bytes of scratch needed (%lld atoms, %d slices of %d x %d), the built-in array holds %zu",
                 need, (long long)n_atoms, p->n_slices, p->nx, p->ny, (size_t)PRISM_STATIC_SCRATCH_BYTES);
        return PRISM_EUNSUPPORTED;
    }
    void* scratch = nullptr;
    CU(potential_static_scratch(&scratch));        // device address of the array on the current device, not its host-side name
    return prism_build_potential(p, atoms_xyz, z_number, n_atoms, luts, n_luts, v, scratch, POT_STATIC_BYTES, cuda_stream);
}

// ---------------------------------------------------------------------------------------------------------
int prism_compute_smatrix(const prism_params* p, const float* v, int32_t* beams_out, void* s,
                          void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    int rc = check_common(p);
    if (rc) return rc;
    if ((rc = check_probe(p))) return rc;
    if (p->f < 1 || p->nx % p->f || p->ny % p->f) return PRISM_EINVAL;
    if (!v || !beams_out || !s || !workspace) return PRISM_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;

    std::vector<int32_t> beams;
    list_beams(p, beams);
    const int n_beams = (int)(beams.size() / 2);
    std::memcpy(beams_out, beams.data(), beams.size() * sizeof(int32_t));

    Arena a(workspace, workspace_bytes);
    SmatrixLayout L;
    layout_smatrix(a, p, n_beams, L);
    if (!a.ok()) return PRISM_ENOMEM;
    DeferredUploads up;
    fill_slice_tables(p, L.tab, up);
    const int xband = band_columns(p), yband = band_rows(p);
    CU(up.flush(st));
    CU(cudaMemcpyAsync(L.beams, beams.data(), beams.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    CU(cudaStreamSynchronize(st));          // the host tables (pageable) are local

    double sigma;
    electron_constants(p->voltage, nullptr, &sigma);
    const size_t npix = (size_t)p->nx * p->ny;
    SliceFeeder& feed = L.feed;
    feed.v = v; feed.on_host = p->potential_on_host != 0; feed.npix = (int64_t)npix; feed.n_slices = p->n_slices;
    feed.sigma = sigma; feed.main_stream = st; feed.pairs = packed_row(p->nx, p->ny);
    if ((rc = feed.init())) { feed.release(); return rc; }

    const int batch = smatrix_batch(p, n_beams);
    const bool s_on_host = p->smatrix_on_host != 0;
    const bool blocked = blocked_grid(p->nx, p->ny);
    // S in host memory: finished layers leave over a private copy stream from one of two alternating
    // buffers (wave batches, or ROW_FINAL staging chunks on blocked grids) while the next batch / chunk is computed
    HostCopyOut out;
    if (s_on_host && (rc = out.init())) { feed.release(); return rc; }
    auto acquire = [&](int i) -> int { return out.acquire(i, st); };
    auto send = [&](int i, void* dst, const void* src, size_t bytes) -> int { return out.send(i, dst, src, bytes, st); };
    auto run = [&]() -> int {
        int n_batch = 0, n_chunk = 0;
        for (int b0 = 0; b0 < n_beams; b0 += batch, ++n_batch) {
            const int nb = std::min(batch, n_beams - b0);
            const int wbuf = L.wave_bufs == 2 ? n_batch % 2 : 0;
            RowArgs ra;
            // S in host memory: the batch is propagated in the workspace and its layers copied out
            ra.a = s_on_host ? L.wave + (size_t)wbuf * batch * npix : (float2*)s + (size_t)b0 * npix;
            ra.out = ra.a; ra.t = feed.tbuf;
            ra.tw_x = L.tab.tw_x; ra.tw_y = L.tab.tw_y; ra.beams = L.beams + b0;
            ra.n_waves = nb; ra.nx = p->nx; ra.ny = p->ny; ra.scale = 1.f; ra.xband = xband;
            ra.blocked = blocked ? 1 : 0;
            ColArgs ca;
            std::memset(&ca, 0, sizeof(ca));
            ca.xband = xband; ca.yband = yband; ca.blocked = ra.blocked;
            ca.a = ra.a; ca.tw_y = L.tab.tw_y; ca.prop_x = L.tab.prop_x; ca.prop_y = L.tab.prop_y;
            ca.ky_lim = L.tab.ky_lim; ca.n_waves = nb; ca.nx = p->nx; ca.ny = p->ny; ca.scale = 1.f;
            int r;
            if (s_on_host && !blocked && (r = acquire(wbuf))) return r;
            feed.begin_sweep();
            for (int sl = 0; sl < p->n_slices; ++sl) {
                if ((r = feed.get(sl))) return r;
                ra.t = feed.current;
                if (sl == 0) {
                    ra.scale = (float)p->nx;                 // keeps A' = nx * FFT_x(t psi), see DESIGN.md
                    LAUNCH(K_ROW_INIT, launch_row_pass(ROW_INIT, ra, st), st);
                } else {
                    LAUNCH(K_ROW_STEP, launch_row_pass(ROW_STEP, ra, st), st);
                }
                LAUNCH(K_COL_STEP, launch_col_pass(COL_STEP, ca, st), st);
            }
            ra.scale = 1.0f / (float)p->nx;
            if (!blocked) {
                LAUNCH(K_ROW_FINAL, launch_row_pass(ROW_FINAL, ra, st), st);
                if (s_on_host && (r = send(wbuf, (float2*)s + (size_t)b0 * npix, ra.a, (size_t)nb * npix * sizeof(float2))))
                    return r;
            } else {
                // blocked mixed space -> natural real space through a staging buffer, a few waves at a time
                for (int c0 = 0; c0 < nb; c0 += L.final_chunk, ++n_chunk) {
                    const int nc = std::min(L.final_chunk, nb - c0);
                    const int sbuf = L.final_bufs == 2 ? n_chunk % 2 : 0;
                    float2* stage = L.final_stage + (size_t)sbuf * L.final_chunk * npix;
                    RowArgs rf = ra;
                    rf.a = ra.a + (size_t)c0 * npix; rf.out = stage; rf.n_waves = nc;
                    if (s_on_host && (r = acquire(sbuf))) return r;
                    LAUNCH(K_ROW_FINAL, launch_row_pass(ROW_FINAL, rf, st), st);
                    if (s_on_host) {
                        if ((r = send(sbuf, (float2*)s + (size_t)(b0 + c0) * npix, stage, (size_t)nc * npix * sizeof(float2))))
                            return r;
                    } else {
                        CU(cudaMemcpyAsync(rf.a, stage, (size_t)nc * npix * sizeof(float2), cudaMemcpyDeviceToDevice, st));
                    }
                }
            }
        }
        // the call's work is complete on `st` only when the last layers have left
        return out.join(st);
    };
    rc = run();
    feed.release();
    return rc;
}

// ---------------------------------------------------------------------------------------------------------
static int copy_out(const prism_params* p, float* out, float* stage, bool out_is_device, cudaStream_t st)
{
    if (out_is_device) return PRISM_OK;
    const size_t bytes = (size_t)p->probes_x * p->probes_y * prism_num_bins(p) * sizeof(float);
    CU(cudaMemcpyAsync(out, stage, bytes, cudaMemcpyDeviceToHost, st));
    return PRISM_OK;
}

// virtual detectors requested beside / instead of the rings: det[probe][d] = sum masks[d] * pattern
struct DetectorRequest { const float* masks = nullptr; int n_masks = 0; float* out = nullptr; };
static int check_detectors(const DetectorRequest& d)
{
    if (!d.out && !d.masks) return PRISM_OK;
    if (!d.out || !d.masks || d.n_masks < 1) return PRISM_EINVAL;
    if (d.n_masks > 16) return PRISM_EUNSUPPORTED;
    if (!pointer_is_device(d.out) || !pointer_is_device(d.masks)) return PRISM_EINVAL;
    return PRISM_OK;
}

// rings (out), full patterns (patterns) and / or virtual detectors (det) of every probe; shared by
// prism_compute_output, prism_compute_patterns and prism_compute_detectors
static int prism_output_impl(const prism_params* p, const void* s, const int32_t* beams, int32_t n_beams,
                             float* out, float* patterns, const DetectorRequest& det,
                             void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    int rc = check_common(p);
    if (rc) return rc;
    if ((rc = check_probe(p))) return rc;
    if ((rc = check_prism(p))) return rc;
    if (!s || !beams || n_beams < 1 || (!out && !patterns && !det.out) || !workspace) return PRISM_EINVAL;
    if (patterns && !pointer_is_device(patterns)) return PRISM_EINVAL;
    if ((rc = check_detectors(det))) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int mx = p->nx / p->f, my = p->ny / p->f, nb = prism_num_bins(p);
    const size_t npix = (size_t)mx * my;
    double lambda;
    electron_constants(p->voltage, &lambda, nullptr);

    Arena a(workspace, workspace_bytes);
    OutputLayout L;
    layout_output(a, p, n_beams, L);
    if (!a.ok()) return PRISM_ENOMEM;
    const bool out_dev = out ? pointer_is_device(out) : true;
    float* d_out = out_dev ? out : L.out_stage;

    // host tables (fp64), uploaded together below
    DeferredUploads up;
    std::vector<float2> h;
    twiddle_table(mx, h);
    up.add(L.tw_x, h);
    std::vector<float2> h2;
    twiddle_table(my, h2);
    up.add(L.tw_y, h2);
    std::vector<int> kxs(n_beams), kys(n_beams);
    std::vector<float2> coef(n_beams);
    const double wscale = 1.0 / (std::sqrt((double)n_beams) * std::sqrt((double)npix));     // R6
    for (int b = 0; b < n_beams; ++b) {
        kxs[b] = beams[2 * b]; kys[b] = beams[2 * b + 1];
        const double qx = kxs[b] / p->cell[0], qy = kys[b] / p->cell[1];
        const double chi = aberration(p, lambda, qx, qy);
        coef[b] = make_float2((float)(wscale * std::cos(-chi)), (float)(wscale * std::sin(-chi)));
    }
    up.add(L.coef_b, coef);
    std::vector<float2> phx, phy;
    position_phases(p->probes_x, p->probe_origin[0], p->probe_step[0], p->cell[0], kxs, phx);
    position_phases(p->probes_y, p->probe_origin[1], p->probe_step[1], p->cell[1], kys, phy);
    up.add(L.phase_x, phx);
    up.add(L.phase_y, phy);
    // window origin (R8): centre = round-half-up pixel, start = centre - M/2, periodic
    std::vector<int> wx0(p->probes_x), wy0(p->probes_y);
    const double px = p->cell[0] / p->nx, py = p->cell[1] / p->ny;
    for (int i = 0; i < p->probes_x; ++i) {
        const long long c = (long long)std::floor((p->probe_origin[0] + i * p->probe_step[0]) / px + 0.5);
        wx0[i] = (int)((((c - mx / 2) % p->nx) + p->nx) % p->nx);
    }
    for (int i = 0; i < p->probes_y; ++i) {
        const long long c = (long long)std::floor((p->probe_origin[1] + i * p->probe_step[1]) / py + 0.5);
        wy0[i] = (int)((((c - my / 2) % p->ny) + p->ny) % p->ny);
    }
    up.add(L.win_x0, wx0);
    up.add(L.win_y0, wy0);
    std::vector<int> bstart, bpix;
    ring_lists(p, mx, my, p->f, p->f, bstart, bpix);
    up.add(L.bin_start, bstart);
    up.add(L.bin_pix, bpix);
    // regular probe lattice: the beam sum of all probes is a Q x Q DFT per S-matrix pixel
    LatticePlan lat = plan_lattice(p, beams, n_beams, wx0, wy0, mx, my);
    const int rows_per_batch = L.batch / p->probes_x;
    if (rows_per_batch < 1) lat.ok = false;
    const bool s_on_host = p->smatrix_on_host != 0;
    if (s_on_host && !lat.ok) return PRISM_EUNSUPPORTED;      // slabs are cut along probe rows of a regular lattice
    std::vector<float2> lcoef;
    if (lat.ok) {
        lcoef.resize(n_beams);
        for (int b = 0; b < n_beams; ++b) {
            const double qx = kxs[b] / p->cell[0], qy = kys[b] / p->cell[1];
            double turns = kxs[b] * (p->probe_origin[0] / p->cell[0]) + kys[b] * (p->probe_origin[1] / p->cell[1]);
            turns -= std::floor(turns);
            const double ang = -aberration(p, lambda, qx, qy) - 2.0 * kPi * turns;
            lcoef[b] = make_float2((float)(wscale * std::cos(ang)), (float)(wscale * std::sin(ang)));
        }
        up.add(L.lat_coef, lcoef);
        up.add(L.cell_beam, lat.cell_beam);
    }
    CU(up.flush(st));
    CU(cudaStreamSynchronize(st));          // host vectors above are local

    const int n_probes = p->probes_x * p->probes_y;
    const int batch = lat.ok ? rows_per_batch * p->probes_x : L.batch;
    SlabRing ring;
    if (s_on_host) {
        ring.s = (const char*)s; ring.slab = (char*)L.slab; ring.cap = L.slab_rows; ring.n_beams = n_beams;
        ring.nx = p->nx; ring.ny = p->ny; ring.my = my; ring.sy = 1 << lat.sy_log2; ring.y00 = wy0[0];
        ring.rows_per_batch = rows_per_batch; ring.probes_y = p->probes_y; ring.main_stream = st;
        if ((rc = ring.init())) { ring.release(); return rc; }
    }
    struct RingGuard { SlabRing& r; ~RingGuard() { r.release(); } } ring_guard{ring};
    for (int p0 = 0; p0 < n_probes; p0 += batch) {
        const int np = std::min(batch, n_probes - p0);
        if (lat.ok) {
            LatticeArgs g;
            g.s = (const float2*)s; g.w = L.w; g.coef = L.lat_coef; g.cell_beam = L.cell_beam;
            g.n_slots = lat.n_slots; g.q = lat.q; g.nx = p->nx; g.ny = p->ny; g.mx = mx; g.my = my;
            g.sx_log2 = lat.sx_log2; g.sy_log2 = lat.sy_log2; g.x00 = wx0[0]; g.y00 = wy0[0];
            g.probes_x = p->probes_x; g.probes_y = p->probes_y;
            g.py0 = p0 / p->probes_x; g.n_rows = np / p->probes_x;
            const int sy = 1 << lat.sy_log2;
            g.row0 = (int)(((long long)g.py0 * sy) % p->ny);
            g.n_pix_rows = std::min(p->ny, sy * (g.n_rows - 1) + my);
            g.slab = 0; g.slab_cap = 0; g.slab_u0 = 0;
            if (s_on_host) {
                const int k = p0 / batch;
                int r;
                if (k == 0 && (r = ring.copy_batch(0))) return r;
                CU(cudaStreamWaitEvent(st, ring.copied[k], 0));
                g.s = L.slab; g.slab = 1; g.slab_cap = ring.cap; g.slab_u0 = ring.u_first(k);
            }
            LAUNCH(K_LATTICE_DFT, launch_lattice_dft(g, st), st);
            if (s_on_host) {
                // the rows of the next batch come in over the copy stream while this batch's windows are transformed
                const int k = p0 / batch;
                CU(cudaEventRecord(ring.done[k], st));
                int r;
                if (p0 + batch < n_probes && (r = ring.copy_batch(k + 1))) return r;
            }
        } else {
            BeamSumArgs g;
            g.s = (const float2*)s; g.w = L.w; g.coef_b = L.coef_b; g.phase_x = L.phase_x; g.phase_y = L.phase_y;
            g.win_x0 = L.win_x0; g.win_y0 = L.win_y0; g.n_beams = n_beams; g.nx = p->nx; g.ny = p->ny;
            g.mx = mx; g.my = my; g.probe0 = p0; g.n_probes_batch = np; g.probes_x = p->probes_x;
            LAUNCH(K_BEAM_SUM, launch_beam_sum(g, st), st);
        }
        // window -> FFT2 -> |.|^2 / (mx my) -> rings, on chip (window_out.cu); the patterns go to HBM only when the
        // caller asked for them or for mask detectors
        WindowArgs wa;
        wa.w = L.w; wa.tw_x = L.tw_x; wa.tw_y = L.tw_y; wa.bin_start = L.bin_start; wa.bin_pix = L.bin_pix;
        wa.out = out ? d_out + (size_t)p0 * nb : nullptr;
        wa.intensity = (patterns || det.out) ? L.intensity : nullptr;
        wa.n = np; wa.mx = mx; wa.my = my; wa.n_bins = nb; wa.scale = (float)(1.0 / (double)npix);
        LAUNCH(K_WINDOW_OUT, launch_window_out(wa, st), st);
        if (patterns)
            LAUNCH(K_PATTERNS, launch_transpose_patterns(L.intensity, patterns + (size_t)p0 * npix, mx, my, np, st), st);
        if (det.out)
            LAUNCH(K_DETECTORS, launch_mask_dot(L.intensity, det.masks, det.n_masks, mx, my,
                                                det.out + (size_t)p0 * det.n_masks, np, st), st);
    }
    return out ? copy_out(p, out, L.out_stage, out_dev, st) : PRISM_OK;
}

int prism_compute_output(const prism_params* p, const void* s, const int32_t* beams, int32_t n_beams,
                         float* out, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (!out) return PRISM_EINVAL;
    return prism_output_impl(p, s, beams, n_beams, out, nullptr, DetectorRequest(), workspace, workspace_bytes, cuda_stream);
}

int prism_compute_patterns(const prism_params* p, const void* s, const int32_t* beams, int32_t n_beams,
                           float* patterns, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (!patterns) return PRISM_EINVAL;
    return prism_output_impl(p, s, beams, n_beams, nullptr, patterns, DetectorRequest(), workspace, workspace_bytes, cuda_stream);
}

int prism_compute_detectors(const prism_params* p, const void* s, const int32_t* beams, int32_t n_beams,
                            const float* masks, int32_t n_masks, float* out,
                            void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (!out || !masks) return PRISM_EINVAL;
    DetectorRequest det;
    det.masks = masks; det.n_masks = n_masks; det.out = out;
    return prism_output_impl(p, s, beams, n_beams, nullptr, nullptr, det, workspace, workspace_bytes, cuda_stream);
}

// ---------------------------------------------------------------------------------------------------------
static int multislice_impl(const prism_params* p, const float* v, float* out, float* patterns,
                           const DetectorRequest& det, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    int rc = check_common(p);
    if (rc) return rc;
    if ((rc = check_probe(p))) return rc;
    if (!v || (!out && !patterns && !det.out) || !workspace) return PRISM_EINVAL;
    if (patterns && !pointer_is_device(patterns)) return PRISM_EINVAL;
    if ((rc = check_detectors(det))) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int nx = p->nx, ny = p->ny, nb = prism_num_bins(p);
    const size_t npix = (size_t)nx * ny;
    double lambda, sigma;
    electron_constants(p->voltage, &lambda, &sigma);

    Arena a(workspace, workspace_bytes);
    MultisliceLayout L;
    layout_multislice(a, p, L, out != nullptr);
    if (!a.ok()) return PRISM_ENOMEM;
    const bool out_dev = out ? pointer_is_device(out) : true;
    float* d_out = out_dev ? out : L.out_stage;

    DeferredUploads up;
    fill_slice_tables(p, L.tab, up);
    // probe spectrum (R4-R6): A_k exp(-i chi_k) * sqrt(nx ny) / sqrt(N_A), with the 1/ny of the
    // unscaled inverse column transform folded in; stored transposed [kx][ky]
    std::vector<float2> ap(npix, make_float2(0.f, 0.f));
    const double qmax = p->alpha / lambda;
    long long n_a = 0;
    for (int sy = 0; sy < ny; ++sy)
        for (int sx = 0; sx < nx; ++sx) {
            const double qx = signed_freq(sx, nx) / p->cell[0], qy = signed_freq(sy, ny) / p->cell[1];
            if (qx * qx + qy * qy <= qmax * qmax) ++n_a;
        }
    if (n_a == 0) return PRISM_EINVAL;
    const double amp = std::sqrt((double)nx * (double)ny) / std::sqrt((double)n_a) / (double)ny;
    for (int sx = 0; sx < nx; ++sx)
        for (int sy = 0; sy < ny; ++sy) {
            const double qx = signed_freq(sx, nx) / p->cell[0], qy = signed_freq(sy, ny) / p->cell[1];
            const double q2 = qx * qx + qy * qy;
            if (q2 <= qmax * qmax) {
                const double chi = aberration(p, lambda, qx, qy);
                ap[(size_t)sx * ny + sy] = make_float2((float)(amp * std::cos(-chi)), (float)(amp * std::sin(-chi)));
            }
        }
    up.add(L.aperture_t, ap);
    std::vector<int> kxs(nx), kys(ny);
    for (int m = 0; m < nx; ++m) kxs[m] = signed_freq(m, nx);
    for (int m = 0; m < ny; ++m) kys[m] = signed_freq(m, ny);
    std::vector<float2> phx, phy;
    position_phases(p->probes_x, p->probe_origin[0], p->probe_step[0], p->cell[0], kxs, phx);
    position_phases(p->probes_y, p->probe_origin[1], p->probe_step[1], p->cell[1], kys, phy);
    up.add(L.phase_x, phx);
    up.add(L.phase_y, phy);
    std::vector<int> bstart, bpix;
    ring_lists(p, nx, ny, 1, 1, bstart, bpix);
    up.add(L.bin_start, bstart);
    up.add(L.bin_pix, bpix);
    CU(up.flush(st));
    CU(cudaStreamSynchronize(st));

    SliceFeeder& feed = L.feed;
    feed.v = v; feed.on_host = p->potential_on_host != 0; feed.npix = (int64_t)npix; feed.n_slices = p->n_slices;
    feed.sigma = sigma; feed.main_stream = st; feed.pairs = packed_row(p->nx, p->ny);
    if ((rc = feed.init())) { feed.release(); return rc; }

    const int n_probes = p->probes_x * p->probes_y;
    const int xband = band_columns(p);
    // the pipelined column pass writes the detector plane for in-band columns only: the rest stays zero (R12)
    if (pipelined_grid(nx, ny))
        CU(cudaMemsetAsync(L.intensity, 0, (size_t)L.waves * npix * sizeof(float), st));
    // resident path: rings only (patterns and mask detectors take the per-pass path, which keeps a batch of patterns)
    const bool resident = multislice_resident(p) && feed.t_slices == p->n_slices && out && !patterns && !det.out;
    auto run_resident = [&]() -> int {
        for (int sl = 0; sl < p->n_slices; ++sl) {          // transmission functions of all slices, once
            int r = feed.get(sl);
            if (r) return r;
        }
        MsResidentArgs g;
        g.psi = L.psi; g.intensity = L.intensity; g.t_stack = feed.tbuf; g.tw = L.tab.tw_x;
        g.prop_x = L.tab.prop_x; g.prop_y = L.tab.prop_y; g.ky_lim = L.tab.ky_lim; g.aperture_t = L.aperture_t;
        g.phase_x = L.phase_x; g.phase_y = L.phase_y; g.bin_start = L.bin_start; g.bin_pix = L.bin_pix; g.out = d_out;
        g.n = nx; g.n_slices = p->n_slices; g.probe0 = 0; g.n_probes = n_probes; g.probes_x = p->probes_x;
        g.n_bins = nb; g.xband = xband; g.yband = band_rows(p); g.slots = L.waves;
        g.scale = (float)((double)ny / (double)nx);
        LAUNCH(K_MS_RESIDENT, launch_ms_resident(g, st), st);
        return PRISM_OK;
    };
    auto run = [&]() -> int {
        for (int p0 = 0; p0 < n_probes; p0 += L.batch) {
            const int np = std::min(L.batch, n_probes - p0);
            ColArgs ca;
            std::memset(&ca, 0, sizeof(ca));
            ca.a = L.psi; ca.intensity = L.intensity; ca.tw_y = L.tab.tw_y; ca.prop_x = L.tab.prop_x;
            ca.prop_y = L.tab.prop_y; ca.ky_lim = L.tab.ky_lim; ca.aperture_t = L.aperture_t;
            ca.phase_x = L.phase_x; ca.phase_y = L.phase_y; ca.probe0 = p0; ca.probes_x = p->probes_x;
            ca.n_waves = np; ca.nx = nx; ca.ny = ny; ca.xband = xband; ca.yband = band_rows(p);
            ca.blocked = blocked_grid(nx, ny) ? 1 : 0;
            ca.scale = (float)((double)ny / (double)nx);      // I = |Psi_S|^2 / (nx ny), see DESIGN.md
            RowArgs ra;
            std::memset(&ra, 0, sizeof(ra));
            ra.a = L.psi; ra.out = L.psi; ra.t = feed.tbuf; ra.tw_x = L.tab.tw_x; ra.tw_y = L.tab.tw_y;
            ra.n_waves = np; ra.nx = nx; ra.ny = ny; ra.scale = 1.f; ra.xband = xband; ra.blocked = ca.blocked;
            LAUNCH(K_COL_MS_INIT, launch_col_pass(COL_MS_INIT, ca, st), st);
            feed.begin_sweep();
            for (int sl = 0; sl < p->n_slices; ++sl) {
                int r = feed.get(sl);
                if (r) return r;
                ra.t = feed.current;
                LAUNCH(K_ROW_STEP, launch_row_pass(ROW_STEP, ra, st), st);
                if (sl == p->n_slices - 1) LAUNCH(K_COL_MS_FINAL, launch_col_pass(COL_MS_FINAL, ca, st), st);
                else LAUNCH(K_COL_STEP, launch_col_pass(COL_STEP, ca, st), st);
            }
            if (patterns)
                LAUNCH(K_PATTERNS, launch_transpose_patterns(L.intensity, patterns + (size_t)p0 * npix, nx, ny, np, st), st);
            if (det.out)
                LAUNCH(K_DETECTORS, launch_mask_dot(L.intensity, det.masks, det.n_masks, nx, ny,
                                                    det.out + (size_t)p0 * det.n_masks, np, st), st);
            if (out)
                LAUNCH(K_BIN_REDUCE, launch_bin_reduce(L.intensity, (int64_t)npix, L.bin_start, L.bin_pix, nb,
                                         d_out + (size_t)p0 * nb, np, st), st);
        }
        return PRISM_OK;
    };
    rc = resident ? run_resident() : run();
    feed.release();
    if (rc) return rc;
    return out ? copy_out(p, out, L.out_stage, out_dev, st) : PRISM_OK;
}

int multislice_compute_output(const prism_params* p, const float* v, float* out,
                              void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (!out) return PRISM_EINVAL;
    return multislice_impl(p, v, out, nullptr, DetectorRequest(), workspace, workspace_bytes, cuda_stream);
}

int multislice_compute_patterns(const prism_params* p, const float* v, float* patterns,
                                void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (!patterns) return PRISM_EINVAL;
    return multislice_impl(p, v, nullptr, patterns, DetectorRequest(), workspace, workspace_bytes, cuda_stream);
}

int multislice_compute_detectors(const prism_params* p, const float* v, const float* masks, int32_t n_masks,
                                 float* out, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (!out || !masks) return PRISM_EINVAL;
    DetectorRequest det;
    det.masks = masks; det.n_masks = n_masks; det.out = out;
    return multislice_impl(p, v, nullptr, nullptr, det, workspace, workspace_bytes, cuda_stream);
}

#pragma GCC visibility pop
}  // extern "C"
