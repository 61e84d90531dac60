/*
 * ORACLE -- TEST INFRASTRUCTURE ONLY.  Not part of the product path.
 *
 * A plain, slow, double-precision CPU direct-scatter gridder: the definition the CUDA library
 * (paper_1003_5575_b200/csrc) is checked against.  It shares no code, header, table or helper
 * with that library and neither side includes the other.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 *
 * What it computes (section 5, Eq. 1, :174-183):
 *     V_grid(u, v) = sum_i f_i(r) * V_i delta(u - u_i, v - v_i)
 * "we compute the distance from the visibility to the centre of a given pixel, and then add the
 * value of f_i(r) V_i to that grid cell" (:181), as a scatter: "For each visibility, the RTS
 * calculated which 2 r_max x 2 r_max patch of pixels it affected, and then added the weighted
 * values to those pixels" (:183).  The GCF f is looked up in an oversampled table (BASELINE.json
 * north_star; readings R1-R16).  Loop order t, b, f; no blocking, no reordering.
 *
 * Pins (tests/test_oracle_pins.py, all -m "not gpu"): P1 unit visibility reproduces the table at
 * every sub-cell shift; P2 linearity; P3 total-sum identity; P4 grid -> inverse FFT -> grid
 * correction vs brute-force direct DFT; P5 brute-force gather restatement (:181, :195);
 * P6 the paper's "around 60 visibilities per pixel" (:183); w-planes and per-baseline tables (row f3)
 * against single-table gridding by linearity.  No function here is "parity unpinned".
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC   (no FMA contraction: every operation
 * below rounds once, in the order written, so the mapping is reproducible bit for bit).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_C_M_PER_S 299792458.0

typedef struct {
    int32_t grid_size;          /* N (even); cell (N/2, N/2) is (u, v) = (0, 0)                 */
    double cell_size;           /* du = dv, wavelengths per cell                                */
    int32_t oversample;         /* O                                                            */
    int32_t n_wplanes;          /* P                                                            */
    const int32_t *support;     /* S_p, taps per axis, p = 0..P-1                               */
    double w_max;               /* wavelengths                                                  */
    int32_t kernel_is_complex;  /* 0: float table; 1: (re, im) float pairs, conj for w < 0      */
    const float *kernel;        /* plane-major; plane p is [S_p O][S_p O] samples               */
    const int32_t *table_index; /* NULL, or [n_time][n_baseline]: the GCF of each baseline, chosen by
                                   the caller instead of by |w| (PAPER.md :73, :179 "a unique GCF for
                                   each visibility").  Out of range: dropped.           */
} oracle_params;

typedef struct {
    int64_t x0, y0;   /* patch origin: cells x0..x0+S-1, y0..y0+S-1 */
    int32_t qx, qy;   /* sub-cell table offsets in [0, O)           */
    int32_t plane;    /* w-plane                                     */
    int32_t conj;     /* use the conjugate table (complex table and w < 0) */
    int32_t support;  /* S of that plane                             */
    int32_t dropped;  /* any tap would fall off the grid             */
} oracle_map_t;

static int64_t floor_div(int64_t a, int64_t b) { /* b > 0 */
    int64_t q = a / b;
    if ((a % b != 0) && (a < 0)) q -= 1;
    return q;
}

/* DESIGN.md reading R5/R6: position rounded half-up to the 1/O sub-cell
 * lattice, patch origin x0 = ceil(x - S/2), table offset q = x0 O - (X - S O / 2). */
static void map_axis(double coord_lambda, const oracle_params *p, int S, int64_t *x0, int32_t *q) {
    const int64_t O = p->oversample;
    double a = coord_lambda / p->cell_size;
    double g = a + (double)(p->grid_size / 2);
    double h = g * (double)O;
    double r = floor(h + 0.5);
    if (!(r > -1.0e15 && r < 1.0e15)) { *x0 = INT64_MIN / 4; *q = 0; return; } /* far off-grid */
    int64_t X = (int64_t)r;
    int64_t A = X - ((int64_t)S * O) / 2;
    int64_t o = floor_div(A + O - 1, O);
    *x0 = o;
    *q = (int32_t)(o * O - A);
}

/* Steps 1-4 of the definition for one (baseline vector in metres, frequency scale s = f / c). */
static oracle_map_t map_one(const oracle_params *p, double u_m, double v_m, double w_m, double s, int64_t tb) {
    oracle_map_t m;
    double ul = u_m * s, vl = v_m * s, wl = w_m * s;
    m.plane = 0;
    int bad_table = 0;
    if (p->table_index) {
        m.plane = p->table_index[tb];
        if (m.plane < 0 || m.plane >= p->n_wplanes) { bad_table = 1; m.plane = 0; }
    } else if (p->n_wplanes > 1) {
        double fp = floor(fabs(wl) / p->w_max * (double)p->n_wplanes);
        m.plane = (fp >= (double)(p->n_wplanes - 1)) ? p->n_wplanes - 1 : (int32_t)fp;
    }
    m.support = p->support[m.plane];
    m.conj = (p->kernel_is_complex && wl < 0.0) ? 1 : 0;
    map_axis(ul, p, m.support, &m.x0, &m.qx);
    map_axis(vl, p, m.support, &m.y0, &m.qy);
    const int64_t N = p->grid_size;
    m.dropped = (bad_table || m.x0 < 0 || m.x0 + m.support > N || m.y0 < 0 || m.y0 + m.support > N) ? 1 : 0;
    return m;
}

static const float *plane_ptr(const oracle_params *p, int plane) {
    size_t off = 0;
    for (int k = 0; k < plane; ++k) {
        size_t e = (size_t)p->support[k] * p->oversample;
        off += e * e * (p->kernel_is_complex ? 2 : 1);
    }
    return p->kernel + off;
}

/* The mapping alone, for the exact-integer check of the CUDA map kernel (pin P8).
 * out is [n_time*n_baseline*n_chan][6] int32: x0, y0, qx, qy, plane | conj<<8, dropped. */
int oracle_map(const oracle_params *p, const double *uvw_m, int32_t n_time, int32_t n_baseline,
               const double *freq_hz, int32_t n_chan, int32_t *out) {
    for (int64_t t = 0; t < n_time; ++t)
        for (int64_t b = 0; b < n_baseline; ++b) {
            const double *L = uvw_m + (t * n_baseline + b) * 3;
            for (int64_t f = 0; f < n_chan; ++f) {
                double s = freq_hz[f] / ORACLE_C_M_PER_S;
                oracle_map_t m = map_one(p, L[0], L[1], L[2], s, t * n_baseline + b);
                int32_t *o = out + ((t * n_baseline + b) * n_chan + f) * 6;
                int64_t cx = m.x0, cy = m.y0;
                if (cx < -(1 << 30)) cx = -(1 << 30);
                if (cx > (1 << 30)) cx = (1 << 30);
                if (cy < -(1 << 30)) cy = -(1 << 30);
                if (cy > (1 << 30)) cy = (1 << 30);
                o[0] = (int32_t)cx; o[1] = (int32_t)cy; o[2] = m.qx; o[3] = m.qy;
                o[4] = m.plane | (m.conj << 8); o[5] = m.dropped;
            }
        }
    return 0;
}

/* Direct scatter restricted to the window rows [y_lo, y_hi) x columns [x_lo, x_hi) of the grid:
 * taps outside the window are skipped, everything else is the definition.  The whole grid is the
 * window (0, N, 0, N).  G (complex128: re, im) and A (float64, may be NULL) point at the window's
 * first cell; cell (pol, y, x) of the window sits at pol*pol_stride + (y-y_lo)*row_pitch + (x-x_lo).
 * A receives sum |w| |V| |k| -- the tolerance denominator of BASELINE.json.  Both are added to.
 * stats[0] += dropped visibilities, stats[1] += sum of S^2 over gridded (not dropped) ones. */
static void scatter_window(const oracle_params *p, const double *uvw_m, int32_t n_time,
                           int32_t n_baseline, const double *freq_hz, int32_t n_chan,
                           const float *vis, const float *weight, int64_t y_lo, int64_t y_hi,
                           int64_t x_lo, int64_t x_hi, int64_t pol_stride, int64_t row_pitch,
                           double *G, double *A, int64_t *stats) {
    const int64_t O = p->oversample;
    const int cplx = p->kernel_is_complex ? 1 : 0;
    int64_t n_drop = 0, n_taps = 0;
    for (int64_t t = 0; t < n_time; ++t)
        for (int64_t b = 0; b < n_baseline; ++b) {
            const double *L = uvw_m + (t * n_baseline + b) * 3;
            for (int64_t f = 0; f < n_chan; ++f) {
                const int64_t i = (t * n_baseline + b) * n_chan + f;
                double s = freq_hz[f] / ORACLE_C_M_PER_S;
                oracle_map_t m = map_one(p, L[0], L[1], L[2], s, t * n_baseline + b);
                if (m.dropped) { n_drop++; continue; }
                const int64_t S = m.support;
                n_taps += S * S;
                if (m.y0 >= y_hi || m.y0 + S <= y_lo || m.x0 >= x_hi || m.x0 + S <= x_lo) continue;
                const float *K = plane_ptr(p, m.plane);
                const int64_t pitch = S * O;
                const double wgt = weight ? (double)weight[i] : 1.0;
                const float *V = vis + i * 8;
                for (int64_t ty = 0; ty < S; ++ty) {
                    const int64_t gy = m.y0 + ty;
                    if (gy < y_lo || gy >= y_hi) continue;
                    for (int64_t tx = 0; tx < S; ++tx) {
                        const int64_t gx = m.x0 + tx;
                        if (gx < x_lo || gx >= x_hi) continue;
                        const int64_t j = (m.qy + ty * O) * pitch + (m.qx + tx * O);
                        double kr, ki;
                        if (cplx) { kr = (double)K[2 * j]; ki = (double)K[2 * j + 1]; if (m.conj) ki = -ki; }
                        else { kr = (double)K[j]; ki = 0.0; }
                        const double kabs = cplx ? sqrt(kr * kr + ki * ki) : fabs(kr);
                        for (int pol = 0; pol < 4; ++pol) {
                            const double vr = wgt * (double)V[2 * pol];
                            const double vi = wgt * (double)V[2 * pol + 1];
                            const int64_t c = pol * pol_stride + (gy - y_lo) * row_pitch + (gx - x_lo);
                            G[2 * c] += vr * kr - vi * ki;
                            G[2 * c + 1] += vr * ki + vi * kr;
                            if (A) A[c] += sqrt(vr * vr + vi * vi) * kabs;
                        }
                    }
                }
            }
        }
    if (stats) { stats[0] += n_drop; stats[1] += n_taps; }
}

/* Several windows, one OpenMP thread per window at a time (each window has exactly one writer, so
 * the result does not depend on the thread count).  win is [n_win][7] = y_lo, y_hi, x_lo, x_hi,
 * offset, pol_stride, row_pitch (the last three in cells): window k writes at G + 2*offset and
 * A + offset.  Row bands of one shared [4][N][N] grid are windows (y_lo, y_hi, 0, N) with
 * offset = y_lo*N, pol_stride = N*N, row_pitch = N.  stats counts once (window 0). */
int oracle_grid_windows(const oracle_params *p, const double *uvw_m, int32_t n_time,
                        int32_t n_baseline, const double *freq_hz, int32_t n_chan, const float *vis,
                        const float *weight, int32_t n_win, const int64_t *win, double *G, double *A,
                        int64_t *stats, int32_t n_threads) {
    if (!p || !uvw_m || !freq_hz || !vis || !G || !win) return -1;
    for (int k = 0; k < n_win; ++k) {
        const int64_t *w = win + 7 * k;
        if (w[0] < 0 || w[2] < 0 || w[1] > p->grid_size || w[3] > p->grid_size || w[1] < w[0] || w[3] < w[2])
            return -1;
    }
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif
#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < n_win; ++k) {
        const int64_t *w = win + 7 * k;
        scatter_window(p, uvw_m, n_time, n_baseline, freq_hz, n_chan, vis, weight, w[0], w[1], w[2],
                       w[3], w[5], w[6], G + 2 * w[4], A ? A + w[4] : NULL, (k == 0) ? stats : NULL);
    }
    return 0;
}

int oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
