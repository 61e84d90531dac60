// The uvw -> (patch origin, sub-cell offset, w-plane) mapping shared by the library's kernels
// (map kernel of gridder_bin, gridder_map, the atomic-scatter gridder).  Not shared with the oracle.
#pragma once
#include "gridder_internal.cuh"

namespace gridder {

// ------------------------------------------------------------------------------------------
// The mapping (steps 1-4).  Every FP64 operation is an explicit
// round-to-nearest intrinsic, so no FMA contraction can change a result: this must agree with the
// definition to the last bit, because one visibility in the wrong sub-cell is far outside the
// tolerance.
// ------------------------------------------------------------------------------------------
struct AxisMap {
    int x0;         // patch origin (clamped to +-2^30 for positions far outside any grid)
    int q;          // sub-cell table offset in [0, O)
    bool far;       // hopelessly off the grid
};

static __device__ __noinline__ void map_axis_wide(double r, int S, int O, int *x0, int *q) {
    // the same algebra in 64 bits, for positions far outside any grid (always dropped, but the
    // test interface reports them)
    const long long X = (long long)r, OO = O;
    const long long A = X - ((long long)S * OO) / 2;
    const long long n = A + OO - 1;
    long long d = n / OO;
    if ((n % OO != 0) && (n < 0)) d -= 1;
    const long long lim = 1ll << 30;
    *x0 = (int)(d < -lim ? -lim : (d > lim ? lim : d));
    *q = (int)(d * OO - A);
}

// Steps 3 of the definition for one axis.  The definition divides by the cell size; a correctly rounded
// FP64 division is ~4x the cost of everything else here, so the position is first computed with a
// multiplication by RN(1 / du).  That value differs from the definition's by less than
// 2^-48 (|h| + N O) (two roundings more, each <= 1 ulp, carried through the same monotone steps), so
// it rounds to the same sub-cell unless h + 0.5 lies within that distance of an integer: only then
// (about one visibility in 10^7, and every exact tie) is the division done.  The result is the
// definition's, bit for bit, by construction -- not "almost always".
__device__ __forceinline__ AxisMap map_axis(double coord_lambda, const MapParams &p, int S) {
    AxisMap m;
    const int O = p.oversample;
    const double half_n = (double)(p.n_grid / 2), dO = (double)O;
    const double h1 = __dmul_rn(__dadd_rn(__dmul_rn(coord_lambda, p.rcp_cell), half_n), dO);
    const double t1 = __dadd_rn(h1, 0.5);
    double r = floor(t1);
    const double fr = t1 - r;                                  // exact (Sterbenz), in [0, 1)
    const double eps = __dadd_rn(__dmul_rn(fabs(h1) + p.span, 3.5527136788005009e-15), 1.0e-30);   // 2^-48
    if (!(fr > eps && fr < 1.0 - eps) || !(fabs(h1) < 1073741824.0)) {
        const double a = __ddiv_rn(coord_lambda, p.cell_size);
        const double g = __dadd_rn(a, half_n);
        const double h = __dmul_rn(g, dO);
        r = floor(__dadd_rn(h, 0.5));
    }
    m.far = false;
    if (r > -1073741824.0 && r < 1073741824.0) {
        // |X| < 2^30 sub-cells (N*O <= 2^21 for every accepted plan): 32-bit integer algebra
        const int X = (int)r;
        const int A = X - ((S * O) >> 1);
        const int n = A + O - 1;              // x0 = ceil(A / O) = floor((A + O - 1) / O)
        int x0;
        if (p.o_shift >= 0) {                 // O a power of two: floor division is an arithmetic shift
            x0 = n >> p.o_shift;
        } else {
            x0 = n / O;
            if ((n % O != 0) && (n < 0)) x0 -= 1;
        }
        m.x0 = x0;
        m.q = x0 * O - A;
    } else if (r > -1.0e15 && r < 1.0e15) {
        map_axis_wide(r, S, O, &m.x0, &m.q);
    } else {
        m.far = true;
        m.x0 = -(1 << 30);
        m.q = 0;
    }
    return m;
}

struct VisMap {
    int x0, y0;     // patch origin, 32-bit (a visibility beyond +-2^30 cells is dropped either way)
    int qx, qy, plane, conj, S;
    bool dropped;
};

__device__ __forceinline__ VisMap map_vis(double u_m, double v_m, double w_m, double s, const MapParams &p,
                                          unsigned int tb = 0) {
    const double ul = __dmul_rn(u_m, s), vl = __dmul_rn(v_m, s);
    VisMap m;
    m.plane = 0;
    m.conj = 0;
    if (p.n_planes > 1 || p.is_complex) {
        const double wl = __dmul_rn(w_m, s);
        if (p.table_index) {
            // (handled below: the caller chose the table)
        } else if (p.n_planes > 1) {
            const double fp = floor(__dmul_rn(__ddiv_rn(fabs(wl), p.w_max), (double)p.n_planes));
            m.plane = (fp >= (double)(p.n_planes - 1)) ? p.n_planes - 1 : (int)fp;
        }
        m.conj = (p.is_complex && wl < 0.0) ? 1 : 0;
    }
    bool bad_table = false;
    if (p.table_index) {           // row f3: per-baseline GCF; an index outside the bank drops the baseline
        const int t = p.table_index[tb];
        bad_table = t < 0 || t >= p.n_planes;
        m.plane = bad_table ? 0 : t;
    }
    m.S = p.support[m.plane];
    const AxisMap mx = map_axis(ul, p, m.S), my = map_axis(vl, p, m.S);
    m.x0 = mx.x0; m.y0 = my.x0; m.qx = mx.q; m.qy = my.q;
    const int N = p.n_grid, S = m.S;
    m.dropped = bad_table || mx.far || my.far || m.x0 < 0 || m.x0 + S > N || m.y0 < 0 || m.y0 + S > N;
    return m;
}

// The production mapper of the pre-summed path: ONE fused multiply-add per axis.  Per channel the scale
// ks = RN(RN(s rcp_cell) O) is formed once (O a power of two: the last product is exact); per visibility and axis
//     t1 = RN(coord_m ks + (N/2 O + 1/2)).
// With H = coord_m s / du O + N/2 O the exact position in sub-cells and u = 2^-53:
//   the definition's t = RN(h + 1/2), h from four roundings, lies within 5.01 u (|H| + N O / 2 + 1) of H + 1/2;
//   t1 (three roundings in ks, one in the FMA) lies within (3.01 |H| + 2.01 N O / 2 + 1) u of it;
// so |t1 - t| < 8.1 u (|H| + N O / 2 + 1) < 2^-48.7 N O for |H| < 2 N O, and floor(t1) = floor(t) whenever t1 is
// farther than eps = 2^-47 N O from every integer -- the same margin FastMap uses, five times the bound.  Anything
// closer (about one visibility in 10^8, and every exact tie) or farther out than 2 N O goes to map_vis: the result
// is the definition's bit for bit by construction.  floor and the distance to the nearest integer come from the
// 1.5 * 2^52 trick: m = RN(t1 + M) holds RN(t1) in its low mantissa bits, d = t1 - (m - M) is exact.
struct FastMap2 {
    double rcp_cell, d_o, chalf, eps, span2;
    int b_off;                                                  // O - 1 - S O / 2
    uint32_t b_lim;                                             // (N - S) O + O - 1: largest b on the grid

    __device__ __forceinline__ void init(const MapParams &p) {
        rcp_cell = p.rcp_cell; d_o = (double)p.oversample;
        chalf = p.fm_chalf;                                     // N/2 O + 1/2
        eps = p.fm_eps;                                         // 2^-47 N O
        span2 = p.fm_span2;
        b_off = p.oversample - 1 - p.fm_half_so;
        b_lim = (uint32_t)(p.fm_n_minus_s * p.oversample + p.oversample - 1);
    }
    __device__ __forceinline__ double chan_scale(double s) const { return __dmul_rn(__dmul_rn(s, rcp_cell), d_o); }
    // LATTICE CODE of the visibility: (by << 16) | bx with b = floor(t) - S O / 2 + O - 1 >= 0, i.e. patch origin
    // x0 = bx / O and offset qx = x0 O + O - 1 - bx -- one word that is equal for two visibilities exactly when
    // their sort keys are (N O <= 46340 on the fast path, so each axis fits 16 bits), and ten integer instructions
    // cheaper to make than the key; key_of() turns it into the key where one is needed (the head of a record).
    // kDropped: off the grid; kUndecided: the screen does not decide, the caller takes slow_lat.
    // Both axes are computed first and tested together: one branch per visibility.
    __device__ __forceinline__ uint32_t lat(double u_m, double v_m, double ks) const {
        const double kMagic = 6755399441055744.0;               // 1.5 * 2^52
        const double tx = __fma_rn(u_m, ks, chalf), ty = __fma_rn(v_m, ks, chalf);
        const double mx = __dadd_rn(tx, kMagic), my = __dadd_rn(ty, kMagic);
        const double dx = __dadd_rn(tx, -__dadd_rn(mx, -kMagic)), dy = __dadd_rn(ty, -__dadd_rn(my, -kMagic));
        if (fabs(tx) < span2 && fabs(ty) < span2 && fabs(dx) > eps && fabs(dy) > eps) {
            // floor(t) = RN(t) - (d < 0): the sign of d is the top bit of its high word
            const int bx = __double2loint(mx) + (__double2hiint(dx) >> 31) + b_off;
            const int by = __double2loint(my) + (__double2hiint(dy) >> 31) + b_off;
            if ((unsigned)bx > b_lim || (unsigned)by > b_lim) return kDropped;       // off the grid
            return ((uint32_t)by << 16) | (uint32_t)bx;
        }
        return kUndecided;                                      // rare: near a rounding boundary, or far away
    }
    // the same from the definition's own mapper (kept out of lat() so that unrolled callers inline it once)
    static __device__ __forceinline__ uint32_t slow_lat(double u_m, double v_m, double s, const MapParams &p) {
        const VisMap m = map_vis(u_m, v_m, 0.0, s, p);
        if (m.dropped) return kDropped;
        const int o = p.oversample;
        return ((uint32_t)(m.y0 * o - m.qy + o - 1) << 16) | (uint32_t)(m.x0 * o - m.qx + o - 1);
    }
    // sort key (fast_key's layout) of a lattice code; `gtile`: first tile id of the visibility's grid
    static __device__ __forceinline__ uint32_t key_of(uint32_t c, const MapParams &p, uint32_t gtile = 0) {
        const uint32_t bx = c & 0xFFFFu, by = c >> 16, om1 = (uint32_t)p.oversample - 1u;
        uint32_t x0, y0;
        if (p.o_shift >= 0) { x0 = bx >> p.o_shift; y0 = by >> p.o_shift; }
        else { x0 = bx / (uint32_t)p.oversample; y0 = by / (uint32_t)p.oversample; }
        const uint32_t qx = x0 * (uint32_t)p.oversample + om1 - bx, qy = y0 * (uint32_t)p.oversample + om1 - by;
        const uint32_t tmask = (1u << p.key.tlog) - 1u;
        const uint32_t tile = gtile + (y0 >> p.key.tlog) * (uint32_t)p.ntx + (x0 >> p.key.tlog);
        return (tile << p.key.tile_shift) | ((y0 & tmask) << (p.key.aux_bits + p.key.tlog)) | ((x0 & tmask) << p.key.aux_bits) |
               (qy << p.key.bits_q) | qx;
    }
    static constexpr uint32_t kUndecided = 0xFFFFFFFEu, kDropped = 0xFFFFFFFDu;     // never lattice codes (nor kAbsent)
};

}  // namespace gridder
