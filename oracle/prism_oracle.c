/*
 * prism_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see prism_oracle.h).
 *
 * fp64 CPU oracle for the PRISM / multislice hot path of arXiv 1706.08563.
 * Each function cites the passage of /root/reference/PAPER.md it follows and,
 * where the paper is silent, the reading (R#) recorded in DESIGN.md.
 * No blocking, fusion or reordering beyond what the cited definition states;
 * OpenMP is used only over independent beams / probes.
 */
#include "prism_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static const double ORC_PI = 3.14159265358979323846264338327950288;

/* ---------- small complex helpers (kept explicit so signs can be read) ---- */
static inline orc_c128 c_make(double re, double im) { orc_c128 z = { re, im }; return z; }
static inline orc_c128 c_add(orc_c128 a, orc_c128 b) { return c_make(a.re + b.re, a.im + b.im); }
static inline orc_c128 c_sub(orc_c128 a, orc_c128 b) { return c_make(a.re - b.re, a.im - b.im); }
static inline orc_c128 c_mul(orc_c128 a, orc_c128 b)
{ return c_make(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re); }
static inline orc_c128 c_expi(double phi) { return c_make(cos(phi), sin(phi)); }
static inline double   c_abs2(orc_c128 a) { return a.re * a.re + a.im * a.im; }

/* signed frequency index of array slot m on an n-point grid (header convention) */
static inline int freq_index(int m, int n) { return m < n / 2 ? m : m - n; }

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------- */
/* O1. Relativistic wavelength and interaction constant.
 * PAPER.md:46 and :80 name sigma ("beam-sample interaction constant") and
 * lambda ("electron wavelength") without formulas; BASELINE.json config 1 says
 * "relativistic lambda, sigma".  Reading R0: the closed forms
 *   lambda = h c / sqrt(eV (2 m c^2 + eV))
 *   sigma  = (2 pi / (lambda V)) (m c^2 + eV) / (2 m c^2 + eV)
 * with CODATA-2018 exact/recommended constants. */
void orc_constants(double voltage, double *lambda, double *sigma)
{
    const double h  = 6.62607015e-34;      /* J s   */
    const double c  = 299792458.0;         /* m / s */
    const double e  = 1.602176634e-19;     /* C     */
    const double me = 9.1093837015e-31;    /* kg    */
    const double ev   = e * voltage;       /* kinetic energy, J */
    const double mc2  = me * c * c;        /* rest energy, J    */
    const double lam_m = h * c / sqrt(ev * (2.0 * mc2 + ev));
    const double lam_a = lam_m * 1e10;     /* Angstrom */
    if (lambda) *lambda = lam_a;
    if (sigma)  *sigma  = (2.0 * ORC_PI / (lam_a * voltage)) * (mc2 + ev) / (2.0 * mc2 + ev);
}

/* ------------------------------------------------------------------------- */
/* Naive O(n^2) DFT, the definition in the header. sign=-1 forward, +1 inverse
 * (unscaled in both directions). The angle is reduced with an exact integer
 * product (k*j mod n) before the call to cos/sin. */
void orc_dft_naive(const orc_c128 *in, orc_c128 *out, int n, int sign)
{
    for (int k = 0; k < n; ++k) {
        orc_c128 acc = c_make(0.0, 0.0);
        for (int j = 0; j < n; ++j) {
            long long kj = ((long long)k * j) % n;
            double phi = sign * 2.0 * ORC_PI * (double)kj / (double)n;
            acc = c_add(acc, c_mul(in[j], c_expi(phi)));
        }
        out[k] = acc;
    }
}

/* Iterative radix-2 decimation-in-time FFT (bit reversal, then log2 n butterfly
 * levels); n must be a power of two.  Unscaled; sign as above.  This is the
 * textbook Cooley-Tukey algorithm; tests pin it to orc_dft_naive and to an
 * independent library FFT. */
void orc_fft(orc_c128 *x, int n, int sign)
{
    /* bit-reversal permutation */
    for (int i = 1, j = 0; i < n; ++i) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { orc_c128 tmp = x[i]; x[i] = x[j]; x[j] = tmp; }
    }
    for (int len = 2; len <= n; len <<= 1) {
        int half = len / 2;
        for (int j = 0; j < half; ++j) {
            orc_c128 w = c_expi(sign * 2.0 * ORC_PI * (double)j / (double)len);
            for (int base = 0; base < n; base += len) {
                orc_c128 u = x[base + j];
                orc_c128 v = c_mul(x[base + j + half], w);
                x[base + j]        = c_add(u, v);
                x[base + j + half] = c_sub(u, v);
            }
        }
    }
}

/* 2-D transform of a[ny][nx]: every row, then every column.
 * sign=-1: forward, unscaled. sign=+1: inverse, divided by nx*ny. */
static void transform2(orc_c128 *a, int ny, int nx, int sign, int use_naive)
{
    int nmax = nx > ny ? nx : ny;
    orc_c128 *line = (orc_c128 *)malloc(sizeof(orc_c128) * (size_t)nmax);
    orc_c128 *res  = (orc_c128 *)malloc(sizeof(orc_c128) * (size_t)nmax);
    for (int y = 0; y < ny; ++y) {
        orc_c128 *row = a + (size_t)y * nx;
        if (use_naive) { orc_dft_naive(row, res, nx, sign); memcpy(row, res, sizeof(orc_c128) * (size_t)nx); }
        else           { orc_fft(row, nx, sign); }
    }
    for (int x = 0; x < nx; ++x) {
        for (int y = 0; y < ny; ++y) line[y] = a[(size_t)y * nx + x];
        if (use_naive) { orc_dft_naive(line, res, ny, sign); memcpy(line, res, sizeof(orc_c128) * (size_t)ny); }
        else           { orc_fft(line, ny, sign); }
        for (int y = 0; y < ny; ++y) a[(size_t)y * nx + x] = line[y];
    }
    if (sign > 0) {
        double inv = 1.0 / ((double)nx * (double)ny);
        for (size_t i = 0; i < (size_t)nx * ny; ++i) { a[i].re *= inv; a[i].im *= inv; }
    }
    free(line); free(res);
}
void orc_fft2(orc_c128 *a, int ny, int nx, int sign)       { transform2(a, ny, nx, sign, 0); }
void orc_dft2_naive(orc_c128 *a, int ny, int nx, int sign) { transform2(a, ny, nx, sign, 1); }

/* ------------------------------------------------------------------------- */
/* O2. Projected potential from a per-species lookup table.
 * PAPER.md:40 "implemented by using a precomputed lookup table for each atom
 * type", :116 "dividing the atomic coordinates into thin slices ... using the
 * cached potentials"; Fig. 1a "All atoms are separated into slices".
 * Readings: R14 slice = floor(z/t) clamped to [0,S-1], whole atom in one slice;
 * R16 sub-pixel exact distance from each pixel centre to the atom; v_Z(r) is the
 * piecewise-linear interpolant of the caller's table on [0, r_cut], 0 beyond
 * (inclusive cut); periodic wrap in x and y. */
static double lut_eval(const double *tab, int n, double r_cut, double r)
{
    double u = r / r_cut * (double)(n - 1);
    int i = (int)floor(u);
    if (i >= n - 1) return tab[n - 1];          /* r == r_cut */
    double w = u - (double)i;
    return tab[i] + w * (tab[i + 1] - tab[i]);
}

int orc_potential(const orc_params *p, const double *atoms_xyz, const int32_t *z,
                  int64_t n_atoms, const int32_t *lut_z, int32_t n_luts,
                  int32_t lut_n, double r_cut, const double *lut_v, double *v)
{
    const int nx = p->nx, ny = p->ny, ns = p->n_slices;
    const double px = p->lx / nx, py = p->ly / ny;
    if (2.0 * r_cut >= p->lx || 2.0 * r_cut >= p->ly) return -2;
    memset(v, 0, sizeof(double) * (size_t)ns * ny * nx);
    for (int64_t a = 0; a < n_atoms; ++a) {
        const double ax = atoms_xyz[3 * a + 0], ay = atoms_xyz[3 * a + 1], az = atoms_xyz[3 * a + 2];
        const double *tab = NULL;
        for (int l = 0; l < n_luts; ++l) if (lut_z[l] == z[a]) tab = lut_v + (size_t)l * lut_n;
        if (!tab) return -1;
        int s = (int)floor(az / p->dz);
        if (s < 0) s = 0;
        if (s > ns - 1) s = ns - 1;
        double *vs = v + (size_t)s * ny * nx;
        int i_lo = (int)ceil((ax - r_cut) / px),  i_hi = (int)floor((ax + r_cut) / px);
        int j_lo = (int)ceil((ay - r_cut) / py),  j_hi = (int)floor((ay + r_cut) / py);
        for (int j = j_lo; j <= j_hi; ++j) {
            for (int i = i_lo; i <= i_hi; ++i) {
                double dx = (double)i * px - ax, dy = (double)j * py - ay;
                double r = sqrt(dx * dx + dy * dy);
                if (r > r_cut) continue;
                int iw = ((i % nx) + nx) % nx, jw = ((j % ny) + ny) % ny;
                vs[(size_t)jw * nx + iw] += lut_eval(tab, lut_n, r_cut, r);
            }
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* O3. Transmission function, Eq. (1): t = exp(i sigma V).
 * Reading R2: not band-limited, |t| = 1. */
void orc_transmission(const double *v_slice, double sigma, int64_t npix, orc_c128 *t)
{
    for (int64_t i = 0; i < npix; ++i) t[i] = c_expi(sigma * v_slice[i]);
}

/* O4. Fresnel propagator, Eq. (2): exp(-i pi lambda |q|^2 t), times
 * the 2/3 band-limit mask of BASELINE.json ("Fresnel propagator with a 2/3
 * band-limit"; reading R1: on the propagator only, strict '<',
 * q_Nyq = min(nx/(2 lx), ny/(2 ly))). */
void orc_propagator(const orc_params *p, double dz, orc_c128 *prop)
{
    double lambda; orc_constants(p->voltage, &lambda, NULL);
    const int nx = p->nx, ny = p->ny;
    double qnx = nx / (2.0 * p->lx), qny = ny / (2.0 * p->ly);
    double qnyq = qnx < qny ? qnx : qny;
    double qcut2 = (2.0 / 3.0 * qnyq) * (2.0 / 3.0 * qnyq);
    for (int my = 0; my < ny; ++my) {
        for (int mx = 0; mx < nx; ++mx) {
            double qx = freq_index(mx, nx) / p->lx, qy = freq_index(my, ny) / p->ly;
            double q2 = qx * qx + qy * qy;
            if (q2 < qcut2) prop[(size_t)my * nx + mx] = c_expi(-ORC_PI * lambda * q2 * dz);
            else            prop[(size_t)my * nx + mx] = c_make(0.0, 0.0);
        }
    }
}

/* O5. One slice: psi <- IFFT2[ P . FFT2[ psi . t ] ]  (Eq. 1 then
 * :80 Eq. 2; :132 "transmitted, followed by a batch FFT, then propagated,
 * followed by a batch inverse FFT"). */
void orc_slice_step(orc_c128 *psi, const orc_c128 *t, const orc_c128 *prop,
                    int ny, int nx, int use_naive)
{
    size_t n = (size_t)ny * nx;
    for (size_t i = 0; i < n; ++i) psi[i] = c_mul(psi[i], t[i]);
    transform2(psi, ny, nx, -1, use_naive);
    for (size_t i = 0; i < n; ++i) psi[i] = c_mul(psi[i], prop[i]);
    transform2(psi, ny, nx, +1, use_naive);
}

/* The slice loop ("These steps are alternated until the electron
 * probe has been propagated through the entire sample"; reading R-O5:
 * propagation after every slice, the last included; equal thickness). */
void orc_multislice_wave(const orc_params *p, const double *v, orc_c128 *psi, int use_naive)
{
    const int nx = p->nx, ny = p->ny;
    size_t n = (size_t)nx * ny;
    double sigma; orc_constants(p->voltage, NULL, &sigma);
    orc_c128 *t    = (orc_c128 *)malloc(sizeof(orc_c128) * n);
    orc_c128 *prop = (orc_c128 *)malloc(sizeof(orc_c128) * n);
    orc_propagator(p, p->dz, prop);
    for (int s = 0; s < p->n_slices; ++s) {
        orc_transmission(v + (size_t)s * n, sigma, (int64_t)n, t);
        orc_slice_step(psi, t, prop, ny, nx, use_naive);
    }
    free(t); free(prop);
}

/* ------------------------------------------------------------------------- */
/* aperture test shared by O6 and O8 (reading R4: hard edge, '<=', fp64 from
 * integer indices): (kx/lx)^2 + (ky/ly)^2 <= (alpha/lambda)^2 */
static int in_aperture(const orc_params *p, double lambda, int kx, int ky)
{
    double qx = kx / p->lx, qy = ky / p->ly;
    double qmax = p->alpha / lambda;
    return qx * qx + qy * qy <= qmax * qmax;
}

/* aberration phase (reading R5): chi(q) = pi lambda |q|^2 C1 + (pi/2) C3 lambda^3 |q|^4, plus (reading R5b) the
 * listed terms (2 pi / lambda) c (lambda |q|)^(n+1) / (n+1) cos(m (phi - angle)), phi = atan2(qy, qx) */
static double chi(const orc_params *p, double lambda, double qx, double qy)
{
    double q2 = qx * qx + qy * qy;
    double x = ORC_PI * lambda * q2 * p->defocus
             + 0.5 * ORC_PI * p->cs * lambda * lambda * lambda * q2 * q2;
    if (p->n_aberr > 0 && p->aberr) {
        double theta = lambda * sqrt(q2), phi = atan2(qy, qx);
        for (int i = 0; i < p->n_aberr; ++i) {
            const orc_aberration *a = &p->aberr[i];
            x += 2.0 * ORC_PI / lambda * a->c * pow(theta, a->n + 1) / (a->n + 1) * cos(a->m * (phi - a->angle));
        }
    }
    return x;
}

int orc_num_aperture(const orc_params *p)
{
    double lambda; orc_constants(p->voltage, &lambda, NULL);
    int count = 0;
    for (int my = 0; my < p->ny; ++my)
        for (int mx = 0; mx < p->nx; ++mx)
            count += in_aperture(p, lambda, freq_index(mx, p->nx), freq_index(my, p->ny));
    return count;
}

/* O6. Converged probe at (xp, yp). PAPER.md:42 "the initial converged probe
 * ... typically as an Airy disk function ... positioned at the desired
 * location"; :86 "coherent wave aberrations such as defocus or spherical
 * aberration".  Psi0[k] = A_k exp(-i chi_k) exp(-2 pi i (kx xp/lx + ky yp/ly));
 * psi0 = sum_k Psi0[k] exp(+2 pi i q_k.r) / (sqrt(N_A) sqrt(nx ny)) so that
 * sum_r |psi0|^2 = 1 (reading R6). */
void orc_probe(const orc_params *p, double xp, double yp, orc_c128 *psi)
{
    double lambda; orc_constants(p->voltage, &lambda, NULL);
    const int nx = p->nx, ny = p->ny;
    int n_a = orc_num_aperture(p);
    for (int my = 0; my < ny; ++my) {
        for (int mx = 0; mx < nx; ++mx) {
            int kx = freq_index(mx, nx), ky = freq_index(my, ny);
            orc_c128 val = c_make(0.0, 0.0);
            if (in_aperture(p, lambda, kx, ky)) {
                double qx = kx / p->lx, qy = ky / p->ly;
                double phase = -chi(p, lambda, qx, qy)
                             - 2.0 * ORC_PI * (qx * xp + qy * yp);
                val = c_expi(phase);
            }
            psi[(size_t)my * nx + mx] = val;
        }
    }
    /* sum_k ... exp(+2 pi i q.r) = (nx ny) * IFFT2; fold the scale */
    orc_fft2(psi, ny, nx, +1);
    double scale = sqrt((double)nx * (double)ny) / sqrt((double)n_a);
    for (size_t i = 0; i < (size_t)nx * ny; ++i) { psi[i].re *= scale; psi[i].im *= scale; }
}

/* ------------------------------------------------------------------------- */
/* O7/O11. Annular detector bins ("an array of annular ring virtual
 * detectors"; BASELINE.json "annular 1-mrad detector bins").  Reading R11:
 * angle = lambda |q| (no arctan), bin = floor(angle / step), half-open rings,
 * pixels with bin >= n_bins dropped, n_bins = round(det_max / det_step). */
int orc_num_bins(const orc_params *p) { return (int)floor(p->det_max / p->det_step + 0.5); }

void orc_bin_intensity(const orc_params *p, const double *intensity, int my_n, int mx_n,
                       int fy, int fx, double *out_bins)
{
    double lambda; orc_constants(p->voltage, &lambda, NULL);
    int nb = orc_num_bins(p);
    for (int b = 0; b < nb; ++b) out_bins[b] = 0.0;
    for (int my = 0; my < my_n; ++my) {
        for (int mx = 0; mx < mx_n; ++mx) {
            double kx = (double)(freq_index(mx, mx_n) * fx);
            double ky = (double)(freq_index(my, my_n) * fy);
            double q = sqrt(kx * kx * (1.0 / (p->lx * p->lx)) + ky * ky * (1.0 / (p->ly * p->ly)));
            double angle = lambda * q;
            int b = (int)floor(angle / p->det_step);
            if (b < nb) out_bins[b] += intensity[(size_t)my * mx_n + mx];
        }
    }
}

/* O6 + O5 + O7.  PAPER.md:132 "the squared intensity of the Fourier transform of
 * the exit wave provides the final result ... at the detector plane".
 * I[k] = |FFT2(psi_S)[k]|^2 / (nx ny). */
void orc_multislice_probe(const orc_params *p, const double *v, double xp, double yp,
                          double *out_bins, double *pattern, int use_naive)
{
    const int nx = p->nx, ny = p->ny;
    size_t n = (size_t)nx * ny;
    orc_c128 *psi = (orc_c128 *)malloc(sizeof(orc_c128) * n);
    double *inten = (double *)malloc(sizeof(double) * n);
    orc_probe(p, xp, yp, psi);
    orc_multislice_wave(p, v, psi, use_naive);
    transform2(psi, ny, nx, -1, use_naive);
    for (size_t i = 0; i < n; ++i) inten[i] = c_abs2(psi[i]) / (double)n;
    orc_bin_intensity(p, inten, ny, nx, 1, 1, out_bins);
    if (pattern) memcpy(pattern, inten, sizeof(double) * n);
    free(psi); free(inten);
}

/* ------------------------------------------------------------------------- */
/* O8. PRISM beams, "every f-th plane wave in both spatial
 * dimensions inside the maximum scattering angle" (reading R7: signed index a
 * multiple of f in both directions, origin included; R4 for the edge).
 * Order: ky ascending over array slots, then kx (array-slot order). */
int orc_beams(const orc_params *p, int32_t *beams, int max_beams)
{
    double lambda; orc_constants(p->voltage, &lambda, NULL);
    int count = 0;
    for (int my = 0; my < p->ny; ++my) {
        for (int mx = 0; mx < p->nx; ++mx) {
            int kx = freq_index(mx, p->nx), ky = freq_index(my, p->ny);
            if (kx % p->f != 0 || ky % p->f != 0) continue;
            if (!in_aperture(p, lambda, kx, ky)) continue;
            if (beams && count < max_beams) { beams[2 * count] = kx; beams[2 * count + 1] = ky; }
            ++count;
        }
    }
    return count;
}

/* O9. One layer of the compact S-matrix, "Each plane wave
 * component is repeatedly transmitted and propagated through each slice ... the
 * complex-valued output wave is stored in real space to form a single layer".
 * psi0[j][i] = exp(+2 pi i (kx i/nx + ky j/ny)); full grid kept (reading R17). */
void orc_smatrix_layer(const orc_params *p, const double *v, int kx, int ky,
                       orc_c128 *layer, int use_naive)
{
    const int nx = p->nx, ny = p->ny;
    for (int j = 0; j < ny; ++j) {
        for (int i = 0; i < nx; ++i) {
            /* exact integer reduction of the phase before cos/sin */
            long long ax = (((long long)kx * i) % nx + nx) % nx;
            long long ay = (((long long)ky * j) % ny + ny) % ny;
            double phi = 2.0 * ORC_PI * ((double)ax / nx + (double)ay / ny);
            layer[(size_t)j * nx + i] = c_expi(phi);
        }
    }
    orc_multislice_wave(p, v, layer, use_naive);
}

void orc_smatrix(const orc_params *p, const double *v, const int32_t *beams, int n_beams,
                 orc_c128 *s, int use_naive)
{
    size_t n = (size_t)p->nx * p->ny;
    #pragma omp parallel for schedule(dynamic, 1)
    for (int b = 0; b < n_beams; ++b)
        orc_smatrix_layer(p, v, beams[2 * b], beams[2 * b + 1], s + (size_t)b * n, use_naive);
}

/* O10 + O11. One PRISM probe.  PAPER.md:86 "For each probe, a subset of all
 * plane waves is cut out around the maximum value of the input STEM probe. The
 * size length of the subset regions is d/f ... multiplying each plane wave
 * subset by the appropriate coefficient and summing all wave subsets";
 * PAPER.md:128 "the modulus squared of its FFT yields the calculation result".
 * Readings R8 (window M = N/f, centre = round-half-up pixel, start = centre -
 * M/2, periodic wrap), R9 (exact probe position in the phase), R6 (scale
 * 1/(sqrt(N_b) sqrt(Mx My)); I = |FFT2_M(w)|^2 / (Mx My)). */
void orc_prism_probe(const orc_params *p, const orc_c128 *s, const int32_t *beams,
                     int n_beams, double xp, double yp, double *out_bins,
                     double *pattern, int use_naive)
{
    /* the whole grid is the band of rows [0, ny) */
    orc_prism_probe_rows(p, s, 0, p->ny, beams, n_beams, xp, yp, out_bins, pattern, use_naive);
}

/* The same probe when only a band of pixel rows of every layer is in memory
 * (storage only, no new reading: at 2048^2 x 1201 beams the whole fp64
 * S-matrix is 80 GB, the 128 rows one probe's window touches are 5 GB).
 * s_rows[b][r][i] holds pixel row (row0 + r) mod ny of layer b, r < n_rows.
 * Returns 0, or -1 (nothing written) if the probe's window leaves the band. */
int orc_prism_probe_rows(const orc_params *p, const orc_c128 *s_rows, int row0, int n_rows,
                         const int32_t *beams, int n_beams, double xp, double yp,
                         double *out_bins, double *pattern, int use_naive)
{
    double lambda; orc_constants(p->voltage, &lambda, NULL);
    const int nx = p->nx, ny = p->ny, f = p->f;
    const int mx_n = nx / f, my_n = ny / f;
    size_t n = (size_t)nx * n_rows, m = (size_t)mx_n * my_n;
    const double px = p->lx / nx, py = p->ly / ny;
    int ic = (int)floor(xp / px + 0.5), jc = (int)floor(yp / py + 0.5);
    for (int j = 0; j < my_n; ++j) {
        int jw = (((jc - my_n / 2 + j) % ny) + ny) % ny;
        if ((((jw - row0) % ny) + ny) % ny >= n_rows) return -1;
    }
    orc_c128 *w = (orc_c128 *)calloc(m, sizeof(orc_c128));
    double *inten = (double *)malloc(sizeof(double) * m);
    for (int b = 0; b < n_beams; ++b) {
        int kx = beams[2 * b], ky = beams[2 * b + 1];
        double qx = kx / p->lx, qy = ky / p->ly;
        double phase = -chi(p, lambda, qx, qy) - 2.0 * ORC_PI * (qx * xp + qy * yp);
        orc_c128 coef = c_expi(phase);
        const orc_c128 *layer = s_rows + (size_t)b * n;
        for (int j = 0; j < my_n; ++j) {
            int jw = (((jc - my_n / 2 + j) % ny) + ny) % ny;
            int jr = (((jw - row0) % ny) + ny) % ny;       /* where pixel row jw sits in the band */
            for (int i = 0; i < mx_n; ++i) {
                int iw = (((ic - mx_n / 2 + i) % nx) + nx) % nx;
                w[(size_t)j * mx_n + i] = c_add(w[(size_t)j * mx_n + i],
                                                c_mul(coef, layer[(size_t)jr * nx + iw]));
            }
        }
    }
    double scale = 1.0 / (sqrt((double)n_beams) * sqrt((double)m));
    for (size_t i = 0; i < m; ++i) { w[i].re *= scale; w[i].im *= scale; }
    transform2(w, my_n, mx_n, -1, use_naive);
    for (size_t i = 0; i < m; ++i) inten[i] = c_abs2(w[i]) / (double)m;
    orc_bin_intensity(p, inten, my_n, mx_n, f, f, out_bins);
    if (pattern) memcpy(pattern, inten, sizeof(double) * m);
    free(w); free(inten);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* Batched drivers: independent probes in parallel ("repeated for
 * the desired probe positions, typically a 2D grid"). xy[probe] = (xp, yp). */
void orc_multislice_probes(const orc_params *p, const double *v, const double *xy,
                           int n_probes, double *out)
{
    int nb = orc_num_bins(p);
    #pragma omp parallel for schedule(dynamic, 1)
    for (int i = 0; i < n_probes; ++i)
        orc_multislice_probe(p, v, xy[2 * i], xy[2 * i + 1], out + (size_t)i * nb, NULL, 0);
}

void orc_prism_probes(const orc_params *p, const orc_c128 *s, const int32_t *beams,
                      int n_beams, const double *xy, int n_probes, double *out)
{
    int nb = orc_num_bins(p);
    #pragma omp parallel for schedule(dynamic, 1)
    for (int i = 0; i < n_probes; ++i)
        orc_prism_probe(p, s, beams, n_beams, xy[2 * i], xy[2 * i + 1],
                        out + (size_t)i * nb, NULL, 0);
}
