/*
 * prism_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of what the PRISM / multislice hot path
 * computes, written from the paper (arXiv 1706.08563, /root/reference/PAPER.md)
 * and the readings listed in DESIGN.md ("Readings of the paper").
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference leg may call this.  It shares no code, header, table or
 * constant generator with the CUDA library under paper_1706_08563_b200/csrc.
 *
 * Conventions (readings R3, R6):
 *   forward DFT  F[k] = sum_n x[n] exp(-2 pi i k n / N)   (no scale)
 *   inverse DFT  x[n] = (1/N) sum_k F[k] exp(+2 pi i k n / N)
 *   signed frequency index of array slot m:  k = m        for m <  N/2
 *                                            k = m - N    for m >= N/2
 *   arrays are row-major [y][x]; lengths in Angstrom, angles in radian,
 *   voltage in volt.
 *
 * Every function is pinned by tests/test_oracle_*.py (see DESIGN.md "Oracle
 * pins"); none is "parity unpinned".
 */
#ifndef PRISM_ORACLE_H
#define PRISM_ORACLE_H

#include <stdint.h>

typedef struct { double re, im; } orc_c128;

/* Parameters of one simulation, the paper's own knobs
 * (cell, pixel size, slice thickness, voltage,
 *  semi-angle, probe step; interpolation factor f). */
/* One term of the aberration function in the (n, m) expansion (reading R5b; "coherent wave
 * aberrations such as defocus or spherical aberration" names the two rotationally symmetric terms, C1 = (1,0)
 * and C3 = (3,0)):  chi += (2 pi / lambda) * c * (lambda |q|)^(n+1) / (n+1) * cos(m (phi - angle)),
 * phi = atan2(q_y, q_x); c in Angstrom, angle in radian. */
typedef struct orc_aberration { int32_t n, m; double c, angle; } orc_aberration;

typedef struct orc_params {
    double  lx, ly, lz;        /* cell (Angstrom)                              */
    int32_t nx, ny;            /* grid (powers of two)                         */
    int32_t n_slices;          /* S                                            */
    double  dz;                /* slice thickness t (Angstrom)                 */
    double  voltage;           /* accelerating voltage (V)                     */
    double  alpha;             /* probe semi-angle (rad)                       */
    double  defocus, cs;       /* C1, C3 (Angstrom)                            */
    int32_t f;                 /* PRISM interpolation factor                   */
    double  det_step, det_max; /* annular bin width / outer angle (rad)        */
    int32_t n_aberr;           /* further aberration terms (may be 0)          */
    const orc_aberration *aberr;
} orc_params;

/* O1  lambda (Angstrom), sigma (rad / (V Angstrom)) */
void   orc_constants(double voltage, double *lambda, double *sigma);

/* own transforms */
void   orc_dft_naive(const orc_c128 *in, orc_c128 *out, int n, int sign);
void   orc_fft(orc_c128 *x, int n, int sign);               /* radix-2, in place, unscaled */
void   orc_fft2(orc_c128 *a, int ny, int nx, int sign);     /* sign=+1 divides by nx*ny    */
void   orc_dft2_naive(orc_c128 *a, int ny, int nx, int sign);

/* O2  projected potential V[s][y][x] (fp64) from per-Z radial tables.
 * lut_v holds n_luts tables of lut_n samples on [0, r_cut]; lut_z their Z.
 * returns 0, or -1 if an atom's Z has no table, -2 if 2 r_cut >= cell. */
int    orc_potential(const orc_params *p, const double *atoms_xyz, const int32_t *z,
                     int64_t n_atoms, const int32_t *lut_z, int32_t n_luts,
                     int32_t lut_n, double r_cut, const double *lut_v, double *v);

/* O3, O4 */
void   orc_transmission(const double *v_slice, double sigma, int64_t npix, orc_c128 *t);
void   orc_propagator(const orc_params *p, double dz, orc_c128 *prop);

/* O5  one slice step, in place. use_naive!=0 swaps the FFT for the O(N^2) DFT */
void   orc_slice_step(orc_c128 *psi, const orc_c128 *t, const orc_c128 *prop,
                      int ny, int nx, int use_naive);
/* all slices of V (fp64 [S][ny][nx]) */
void   orc_multislice_wave(const orc_params *p, const double *v, orc_c128 *psi, int use_naive);

/* O6  probe in real space, sum |psi|^2 = 1 */
int    orc_num_aperture(const orc_params *p);
void   orc_probe(const orc_params *p, double xp, double yp, orc_c128 *psi);

/* O7 / O11 detector bins */
int    orc_num_bins(const orc_params *p);
/* intensity[ky][kx] on an my x mx grid whose frequencies are k*fx/lx, k*fy/ly */
void   orc_bin_intensity(const orc_params *p, const double *intensity, int my, int mx,
                         int fy, int fx, double *out_bins);

/* O6+O5+O7  one multislice probe -> bins (and, if not NULL, the N x N pattern) */
void   orc_multislice_probe(const orc_params *p, const double *v, double xp, double yp,
                            double *out_bins, double *pattern, int use_naive);

/* O8  beams: returns count; if beams!=NULL fills up to max_beams (kx,ky) pairs */
int    orc_beams(const orc_params *p, int32_t *beams, int max_beams);
/* O9  one S-matrix layer */
void   orc_smatrix_layer(const orc_params *p, const double *v, int kx, int ky,
                         orc_c128 *layer, int use_naive);
/* all layers, OpenMP over beams */
void   orc_smatrix(const orc_params *p, const double *v, const int32_t *beams, int n_beams,
                   orc_c128 *s, int use_naive);
/* O10+O11  one PRISM probe -> bins (and, if not NULL, the M x M pattern) */
void   orc_prism_probe(const orc_params *p, const orc_c128 *s, const int32_t *beams,
                       int n_beams, double xp, double yp, double *out_bins,
                       double *pattern, int use_naive);
/* the same with only pixel rows [row0, row0 + n_rows) (mod ny) of every layer in memory:
 * s_rows[b][r][i] = layer b, pixel row (row0 + r) mod ny.  -1 if the window leaves the band. */
int    orc_prism_probe_rows(const orc_params *p, const orc_c128 *s_rows, int row0, int n_rows,
                            const int32_t *beams, int n_beams, double xp, double yp,
                            double *out_bins, double *pattern, int use_naive);

/* batched drivers (OpenMP over probes); out[probe][bin] */
void   orc_multislice_probes(const orc_params *p, const double *v, const double *xy,
                             int n_probes, double *out);
void   orc_prism_probes(const orc_params *p, const orc_c128 *s, const int32_t *beams,
                        int n_beams, const double *xy, int n_probes, double *out);
int    orc_num_threads(void);

#endif
