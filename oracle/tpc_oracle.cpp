/*
 * tpc_oracle.cpp -- CPU ORACLE for the TPC sector-tracker hot path.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load this.
 * It shares no code, header, table or helper with the CUDA path (paper_1712_09416_b200/csrc) and neither
 * includes the other.  Plain, slow, scalar: every neighbour / candidate search is a linear scan of the row.
 *
 * What the path is: "our TPC tracker ... bases on a Cellular Automaton and on the Kalman filter"
 * (abstract; section 2).  PAPER.md gives no equation for it; the step list is
 * BASELINE.json:5 (north_star): neighbour finding between adjacent pad rows, neighbour cleaning, start-hit
 * selection, Kalman-filter tracklet construction with state (y, z, sin phi, tg lambda, q/pT) in sector-local
 * coordinates, tracklet selection resolving shared hits.  Every detail below is the reading O1..O7 of
 * SURVEY.md 8(c).2, restated with its formulas in DESIGN.md "The method, step by step"; this is an
 * algorithm (a heuristic plus an extended-Kalman iteration), so the oracle follows it step by step.
 *
 * Precision: template<real>.  real = double is the reference arithmetic (pins, margins).  real = float is
 * the strict-float32 mode: BASELINE.json:5 fixes float32 for the fit, and wherever floating point decides an
 * integer (a link, a gate, an arg min) both sides must decide in the same precision; in that mode every
 * expression is evaluated exactly as parenthesised here, IEEE round-to-nearest, no contraction
 * (compile with -ffp-contract=off), only + - * / sqrt.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): O2 against an independent brute-force triplet search and the
 * mirror symmetry; O3/O4 invariants; transport against the closed-form helix and its Jacobian against central
 * differences; fit against the textbook straight-line least squares (Bz -> 0), against noise-free helices,
 * pulls / chi2 per ndf / Gluckstern curvature resolution with noise; O6 ownership invariants and a brute-force
 * owner; end-to-end efficiency on generated events; O8 (refit of the selected tracks) against the
 * generated helix, the least-squares line, a test-side composition of the pinned transport / update steps,
 * chi2 per ndf and Gluckstern (tests/test_oracle_refit.py); O5 search / gate / construct against a Python
 * restatement of DESIGN.md "O5" that drives only the pinned transport / update, and against hand-built sectors
 * with hand-written expected tables for every branch: window edges and clamps, ties, gap counting, edge stop,
 * rejected links, removed hits (tests/test_oracle_constructor.py); O9 against generator truth, a restatement with
 * the exact helix, and hand-built segments on every tie and cut edge (tests/test_oracle_merge.py).
 * PARITY UNPINNED: the exact link / track values on the BASELINE.json configs have no outside reference
 * (the paper prints none); they are pinned only through the properties above.
 */
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {
/* The oracle's own parameter block (same fields as the boundary's tpc_params, declared independently). */
typedef struct {
    int32_t link_step;          /* Delta: neighbour rows r +- Delta (1 or 2) */
    float nf_slope_y, nf_slope_z; /* T_y, T_z: window half width = T*|dx| + w0 */
    float nf_w0;                /* cm */
    float nf_dmax;              /* D_max cm^2 */
    float sin_max;              /* s_max: transport fails beyond */
    float var_s, var_t, var_q;  /* prior variances V_s, V_t, V_q */
    float chi2_link, chi2_ext;  /* 2-dof gates */
    float win_nsigma, win_min, win_max; /* search window n_w, w_min, w_max */
    int32_t max_gap;            /* rows without a hit before a pass ends */
    float edge_margin;          /* cm beyond the wedge before a pass ends */
    int32_t min_tracklet_hits, min_track_hits;
    int32_t refit;              /* O8: 1 = track parameters from a refit over the final hit list */
    int32_t merge;              /* O9: 1 = link track segments across sector borders (needs refit) */
    float merge_dy, merge_dz;   /* cm: tolerated |dy|, |dz| between the extrapolated and the found segment */
    float merge_ds, merge_dt;   /* tolerated |d sin phi|, |d tg lambda| */
    int32_t merge_max_gap;      /* pad rows that may be missing between the two segments */
    int32_t seed_dedup;         /* O5: 1 = a start hit already recorded by the up pass of an earlier tracklet of its
                                 * sector is skipped (no tracklet is built from it); reading R23 */
    int32_t checked;            /* 1 = reject non-finite y / z (the oracle is given no x); S23 */
} oracle_params;

typedef struct {
    int32_t n_sectors, n_rows;
    const float* row_x;         /* [n_rows] */
    float tan_half_angle;
    float sigma_y, sigma_z;
    float bz;
} oracle_geometry;
}

namespace {

constexpr double kLight = 0.00299792458; /* cm^-1 GeV T^-1 */
constexpr double kTiny = 1e-30;

/* smallest relative margin of all float decisions taken for one unit (a hit in O2, a tracklet in O5) */
struct Margin {
    double m = std::numeric_limits<double>::infinity();
    void rel(double a, double b) {
        double d = std::fabs(a - b) / std::max(std::max(std::fabs(a), std::fabs(b)), kTiny);
        if (d < m) m = d;
    }
};
template <class R> inline bool le(R a, R b, Margin& mg) { mg.rel((double)a, (double)b); return a <= b; }
template <class R> inline bool gt(R a, R b, Margin& mg) { mg.rel((double)a, (double)b); return a > b; }

template <class R> struct Fit {
    R y, z, s, t, q;   /* state at x: y, z, sin phi, dz/dS = tg lambda, q/pT */
    R C[5][5];         /* symmetric covariance */
    R chi2;
    int n;             /* hits in the fit */
};

struct Tracklet {
    int32_t first_row = -1, last_row = -1, n_hits = 0;   /* n_hits = 0: no tracklet was built (O5 seed de-duplication) */
    double par[5] = {0, 0, 0, 0, 0};
    double cov[5] = {0, 0, 0, 0, 0}; /* diagonal of the covariance at x_ref */
    double chi2 = 0;
    double margin = std::numeric_limits<double>::infinity();
    std::vector<int32_t> table; /* [n_rows] event-local hit index or -1 */
};

struct Result {
    int32_t n_clusters = 0, n_sectors = 0, n_rows = 0;
    std::vector<int32_t> link_up, link_dn, clink_up, clink_dn; /* [N] event-local index of the neighbour */
    std::vector<double> nf_margin;                              /* [N] */
    std::vector<int32_t> seed_offset;                           /* [n_sectors+1] */
    std::vector<int32_t> start_hit;                             /* [S] canonical order */
    std::vector<Tracklet> tracklets;                            /* [S] */
    /* tracks */
    std::vector<int32_t> trk_sector, trk_first_hit, trk_n_hits, trk_ndf, trk_seed, trk_first_row;
    std::vector<double> trk_x, trk_y, trk_z, trk_sinphi, trk_tgl, trk_qpt, trk_chi2, trk_margin;
    std::vector<int32_t> hit_idx;
    /* O8 outer state (up pass of the refit, at its top hit) and O9 links */
    std::vector<int32_t> trk_row_out, trk_next, trk_prev, trk_global; /* global: first segment of the chain */
    std::vector<double> trk_out; /* [T][6] x y z sin phi tg lambda q/pT */
    std::vector<double> trk_merge_margin; /* [T] smallest relative margin of the O9 decisions a segment took part in */
    /* O10: fit of the global track (chain of linked segments), stored at the chain's first segment; zero elsewhere */
    std::vector<double> trk_g;            /* [T][7] x y z sin phi tg lambda q/pT chi2, in the frame of trk_g_sector */
    std::vector<int32_t> trk_g_ndf, trk_g_n_hits, trk_g_sector;
};

template <class R> struct Sector {
    const oracle_params& P;
    const oracle_geometry& G;
    const float *gy, *gz;  /* event arrays */
    const int32_t* grow;
    int n_rows;
    R kB;                  /* kappa = kB * q */
    std::vector<R> X;      /* row_x as real */
    std::vector<std::vector<int32_t>> rows; /* O1: hits of each row, ascending original index */

    Sector(const oracle_params& p, const oracle_geometry& g, const float* y, const float* z, const int32_t* row)
        : P(p), G(g), gy(y), gz(z), grow(row), n_rows(g.n_rows) {
        kB = R(-1) * (R(kLight) * R(g.bz)); /* kB = -K*Bz */
        X.resize(n_rows);
        for (int r = 0; r < n_rows; r++) X[r] = R(g.row_x[r]);
        rows.resize(n_rows);
    }

    /* ---- O1 bucket ---- */
    void bucket(int32_t begin, int32_t end) {
        for (int32_t h = begin; h < end; h++) rows[grow[h]].push_back(h);
    }

    /* ---- O2 neighbour finder: best (up, down) pair by straight-line deviation ---- */
    void neighbours(Result& res) {
        const int D = P.link_step;
        const R Ty = R(P.nf_slope_y), Tz = R(P.nf_slope_z), w0 = R(P.nf_w0), Dmax = R(P.nf_dmax);
        std::vector<int32_t> U, Dn;
        for (int r = 0; r < n_rows; r++) {
            if (r - D < 0 || r + D >= n_rows) continue;
            const R x0 = X[r], x1 = X[r + D], x2 = X[r - D];
            const R wyu = Ty * std::fabs(x1 - x0) + w0, wzu = Tz * std::fabs(x1 - x0) + w0;
            const R wyd = Ty * std::fabs(x2 - x0) + w0, wzd = Tz * std::fabs(x2 - x0) + w0;
            const R a = (x0 - x2) / (x1 - x2);
            for (int32_t h : rows[r]) {
                Margin mg;
                const R y0 = R(gy[h]), z0 = R(gz[h]);
                U.clear(); Dn.clear();
                for (int32_t u : rows[r + D]) {
                    bool iy = le(std::fabs(R(gy[u]) - y0), wyu, mg);
                    bool iz = le(std::fabs(R(gz[u]) - z0), wzu, mg);
                    if (iy && iz) U.push_back(u);
                }
                for (int32_t d : rows[r - D]) {
                    bool iy = le(std::fabs(R(gy[d]) - y0), wyd, mg);
                    bool iz = le(std::fabs(R(gz[d]) - z0), wzd, mg);
                    if (iy && iz) Dn.push_back(d);
                }
                int32_t bu = -1, bd = -1;
                R best = 0, second = 0;
                bool have = false, have2 = false;
                for (int32_t u : U)          /* ascending u, then ascending d: strict < keeps the lowest pair */
                    for (int32_t d : Dn) {
                        const R yd = R(gy[d]), zd = R(gz[d]);
                        const R yh = yd + a * (R(gy[u]) - yd);
                        const R zh = zd + a * (R(gz[u]) - zd);
                        const R dy = y0 - yh, dz = z0 - zh;
                        const R dev = dy * dy + dz * dz;
                        if (!have || dev < best) {
                            if (have) { second = best; have2 = true; }
                            best = dev; bu = u; bd = d; have = true;
                        } else if (!have2 || dev < second) { second = dev; have2 = true; }
                    }
                if (have2) mg.rel((double)best, (double)second);
                if (have && le(best, Dmax, mg)) { res.link_up[h] = bu; res.link_dn[h] = bd; }
                res.nf_margin[h] = mg.m;
            }
        }
    }

    /* ---- O3 cleaner: keep reciprocal links only (one simultaneous pass) ---- */
    void clean(Result& res, int32_t begin, int32_t end) {
        for (int32_t h = begin; h < end; h++) {
            const int32_t u = res.link_up[h], d = res.link_dn[h];
            res.clink_up[h] = (u >= 0 && res.link_dn[u] == h) ? u : -1;
            res.clink_dn[h] = (d >= 0 && res.link_up[d] == h) ? d : -1;
        }
    }

    /* ---- O4 start hits, ordered by (row, original index) ---- */
    void start_hits(const Result& res, std::vector<int32_t>& out) {
        for (int r = 0; r < n_rows; r++)
            for (int32_t h : rows[r])
                if (res.clink_up[h] >= 0 && res.clink_dn[h] < 0) out.push_back(h);
    }

    /* ---- O5 helpers ---- */
    void prior(Fit<R>& f) const {
        for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) f.C[i][j] = R(0);
        f.C[0][0] = R(G.sigma_y) * R(G.sigma_y);
        f.C[1][1] = R(G.sigma_z) * R(G.sigma_z);
        f.C[2][2] = R(P.var_s); f.C[3][3] = R(P.var_t); f.C[4][4] = R(P.var_q);
        f.chi2 = R(0);
    }

    /* move the fit from x to x1 along the helix; false (fit untouched) if |sin phi| exceeds s_max at either end
       (an update can push sin phi itself past the limit, and sqrt(1 - s^2) must stay real) */
    bool transport(Fit<R>& f, R x, R x1, Margin& mg) const {
        const R dx = x1 - x;
        const R kap = kB * f.q;
        const R s = f.s, s1 = s + kap * dx;
        if (gt(std::fabs(s), R(P.sin_max), mg)) return false;
        if (gt(std::fabs(s1), R(P.sin_max), mg)) return false;
        const R c0 = std::sqrt(R(1) - s * s), c1 = std::sqrt(R(1) - s1 * s1);
        const R icc = R(1) / (c0 + c1), ic0 = R(1) / c0, ic1 = R(1) / c1;
        const R dy = dx * ((s + s1) * icc);
        const R dl2 = dx * dx + dy * dy;
        const R dl = (dx < R(0)) ? -std::sqrt(dl2) : std::sqrt(dl2); /* signed chord */
        const R idl = R(1) / dl;
        const R u = kap * dl, u2 = u * u;
        const R c24 = R(1) / R(24), c640 = R(3) / R(640), c12 = R(1) / R(12);
        const R dS = dl * (R(1) + u2 * (c24 + u2 * c640)); /* arc from chord, series of (2/k) asin(k dl/2) */
        const R ccd = R(1) + (c0 * c1 + s * s1);
        /* Jacobian, rows (y z s t q); identity elsewhere */
        const R Fys = dx * ccd * icc * ic0 * ic1;
        const R Fyq = kB * (dx * dx) * ccd * ic1 * icc * icc;
        const R Fzs = f.t * dy * ic0 * ic1;
        const R Fzt = dS;
        const R Fzq = f.t * ((dy * idl) * Fyq + (kB * kap) * (dl * dl2) * c12);
        const R Fsq = kB * dx;
        R F[5][5];
        for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) F[i][j] = (i == j) ? R(1) : R(0);
        F[0][2] = Fys; F[0][4] = Fyq; F[1][2] = Fzs; F[1][3] = Fzt; F[1][4] = Fzq; F[2][4] = Fsq;
        f.y = f.y + dy; f.z = f.z + f.t * dS; f.s = s1;
        /* C <- F C F^T : M = F C (k ascending), then lower triangle of M F^T (l ascending), mirrored */
        R M[5][5];
        for (int i = 0; i < 5; i++)
            for (int l = 0; l < 5; l++) {
                R acc = R(0);
                for (int k = 0; k < 5; k++) acc = acc + F[i][k] * f.C[k][l];
                M[i][l] = acc;
            }
        for (int i = 0; i < 5; i++)
            for (int j = 0; j <= i; j++) {
                R acc = R(0);
                for (int l = 0; l < 5; l++) acc = acc + M[i][l] * F[j][l];
                f.C[i][j] = acc; f.C[j][i] = acc;
            }
        return true;
    }

    /* ---- O10: the fit, given at x in the frame of one sector, expressed in the frame of a neighbouring sector, whose
       axis is turned by the angle with sine sn and cosine cd (sn < 0: the next sector in azimuth).  The reference
       point stays the same point of space; its new abscissa x' is returned in x.  Parameters:
         x' = x cd - y sn, y' = x sn + y cd, s' = s cd + sqrt(1 - s^2) sn; z, t, q unchanged.
       Covariance C' = J C J^T with the first-order change of the parameters AT THE PLANE x' = const (a shift dy of
       the point leaves that plane by -sn dy, and is brought back along the track over dl = sn dy / c'):
         dy'/dy = cd + sn s'/c',  dz'/dy = t sn / c',  ds'/dy = kappa sn,  ds'/ds = cd - (s/c) sn,  identity elsewhere.
       false (fit untouched) if |sin phi| exceeds s_max before or after. */
    bool rotate(Fit<R>& f, R& x, R sn, R cd, Margin& mg) const {
        const R s = f.s;
        if (gt(std::fabs(s), R(P.sin_max), mg)) return false;
        const R c = std::sqrt(R(1) - s * s);
        const R s1 = s * cd + c * sn;
        if (gt(std::fabs(s1), R(P.sin_max), mg)) return false;
        const R c1 = std::sqrt(R(1) - s1 * s1);
        const R ic1 = R(1) / c1;
        const R kap = kB * f.q;
        const R Jyy = cd + sn * (s1 * ic1);
        const R Jzy = (f.t * sn) * ic1;
        const R Jsy = kap * sn;
        const R Jss = cd - (s * (R(1) / c)) * sn;
        const R x1 = x * cd - f.y * sn, y1 = x * sn + f.y * cd;
        x = x1; f.y = y1; f.s = s1;
        R J[5][5];
        for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) J[i][j] = (i == j) ? R(1) : R(0);
        J[0][0] = Jyy; J[1][0] = Jzy; J[2][0] = Jsy; J[2][2] = Jss;
        R M[5][5];
        for (int i = 0; i < 5; i++)
            for (int l = 0; l < 5; l++) {
                R acc = R(0);
                for (int k = 0; k < 5; k++) acc = acc + J[i][k] * f.C[k][l];
                M[i][l] = acc;
            }
        for (int i = 0; i < 5; i++)
            for (int j = 0; j <= i; j++) {
                R acc = R(0);
                for (int l = 0; l < 5; l++) acc = acc + M[i][l] * J[j][l];
                f.C[i][j] = acc; f.C[j][i] = acc;
            }
        return true;
    }

    /* ---- O10 fit of a global track: the chain of linked segments seg[0..m) (hit lists row-ascending, at least 2 hits
       in seg[0]), each in its own sector sec[k]; sn_up[k], k >= 1: sine of the turn from sector sec[k-1] to sec[k].
       Up pass as O8 through seg[0]; at the top hit of a segment the fit is turned into the next segment's frame
       (rotate), moved in ONE step to the row of that segment's first hit, updated with it, and goes on row by row.
       Down pass: fresh fit at the last hit the up pass used, (s, t, q) from there, prior covariance, the same way
       back.  A failed transport or rotation ends a pass.  Result: state after the last update of the down pass, in
       the frame of the sector where it ended. */
    bool global_fit(const std::vector<const std::vector<int32_t>*>& seg, const std::vector<R>& sn_up, R cd, double g[7],
                    int& n_fit, int& end_seg) const {
        const int m = (int)seg.size();
        Margin mg;
        Fit<R> f, snap;
        const std::vector<int32_t>& h0 = *seg[0];
        if (h0.size() < 2) return false;
        {
            const R dx = X[grow[h0[1]]] - X[grow[h0[0]]];
            const R dy = R(gy[h0[1]]) - R(gy[h0[0]]), dz = R(gz[h0[1]]) - R(gz[h0[0]]);
            const R dl = std::sqrt(dx * dx + dy * dy);
            f.y = R(gy[h0[0]]); f.z = R(gz[h0[0]]); f.s = dy / dl; f.t = dz / dl; f.q = R(0);
            prior(f); f.n = 1;
        }
        snap = f;
        int k_top = 0, j_top = 0;                 /* segment / position of the last hit the up pass used */
        {
            R xc = X[grow[h0[0]]];
            bool alive = true;
            for (int k = 0; k < m && alive; k++) {
                const std::vector<int32_t>& hk = *seg[k];
                int j = 0;
                if (k == 0) j = 1;
                else {   /* into the frame of segment k, then to the row of its first hit */
                    if (!rotate(f, xc, sn_up[k], cd, mg)) break;
                    const R xb = X[grow[hk[0]]];
                    if (xb != xc && !transport(f, xc, xb, mg)) break;
                    xc = xb;
                    update(f, hk[0]); snap = f; k_top = k; j_top = 0; j = 1;
                }
                for (int row = grow[hk[j - 1]] + 1; j < (int)hk.size() && row <= grow[hk.back()]; row++) {
                    if (!transport(f, xc, X[row], mg)) { alive = false; break; }
                    xc = X[row];
                    if (row == grow[hk[j]]) { update(f, hk[j]); snap = f; k_top = k; j_top = j; j++; }
                }
            }
        }
        {
            const int32_t ht = (*seg[k_top])[j_top];
            f.y = R(gy[ht]); f.z = R(gz[ht]); f.s = snap.s; f.t = snap.t; f.q = snap.q;
            prior(f); f.n = 1;
            snap = f;
            int ref_row = grow[ht];
            end_seg = k_top;
            R xc = X[grow[ht]];
            bool alive = true;
            for (int k = k_top; k >= 0 && alive; k--) {
                const std::vector<int32_t>& hk = *seg[k];
                int j = (k == k_top) ? j_top - 1 : (int)hk.size() - 1;
                if (k < k_top) {   /* back into the frame of segment k, then to the row of its top hit */
                    if (!rotate(f, xc, R(0) - sn_up[k + 1], cd, mg)) break;
                    const R xb = X[grow[hk[j]]];
                    if (xb != xc && !transport(f, xc, xb, mg)) break;
                    xc = xb;
                    update(f, hk[j]); snap = f; ref_row = grow[hk[j]]; end_seg = k; j--;
                }
                for (int row = grow[hk[j + 1]] - 1; j >= 0 && row >= grow[hk[0]]; row--) {
                    if (!transport(f, xc, X[row], mg)) { alive = false; break; }
                    xc = X[row];
                    if (row == grow[hk[j]]) { update(f, hk[j]); snap = f; ref_row = row; end_seg = k; j--; }
                }
            }
            g[0] = (double)X[ref_row];
        }
        g[1] = (double)snap.y; g[2] = (double)snap.z; g[3] = (double)snap.s; g[4] = (double)snap.t; g[5] = (double)snap.q;
        g[6] = (double)snap.chi2; n_fit = snap.n;
        return true;
    }

    /* gate value of a measurement against the predicted state (both variances from the pre-update C) */
    R gate(const Fit<R>& f, R my, R mz) const {
        const R ry = my - f.y, rz = mz - f.z;
        const R wy = R(1) / (f.C[0][0] + R(G.sigma_y) * R(G.sigma_y));
        const R wz = R(1) / (f.C[1][1] + R(G.sigma_z) * R(G.sigma_z));
        return (ry * ry) * wy + (rz * rz) * wz;
    }

    /* one scalar Kalman update with measurement m of state component k (0 = y, 1 = z) */
    void update1(Fit<R>& f, int k, R m, R var) const {
        R* x[5] = {&f.y, &f.z, &f.s, &f.t, &f.q};
        const R r = m - *x[k];
        const R w = R(1) / (f.C[k][k] + var);
        R ck[5], K[5];
        for (int j = 0; j < 5; j++) { ck[j] = f.C[j][k]; K[j] = ck[j] * w; }
        for (int j = 0; j < 5; j++) *x[j] = *x[j] + K[j] * r;
        for (int i = 0; i < 5; i++)
            for (int j = 0; j <= i; j++) {
                const R v = f.C[i][j] - K[i] * ck[j];
                f.C[i][j] = v; f.C[j][i] = v;
            }
        f.chi2 = f.chi2 + (r * r) * w;
    }
    void update(Fit<R>& f, int32_t h) const {
        update1(f, 0, R(gy[h]), R(G.sigma_y) * R(G.sigma_y));
        update1(f, 1, R(gz[h]), R(G.sigma_z) * R(G.sigma_z));
        f.n++;
    }

    /* best hit of a row inside the window of the predicted state; -1 if none passes chi2_ext */
    int32_t search(const Fit<R>& f, int row, Margin& mg) const {
        const R sy2 = R(G.sigma_y) * R(G.sigma_y), sz2 = R(G.sigma_z) * R(G.sigma_z);
        const R wy = std::min(std::max(R(P.win_nsigma) * std::sqrt(f.C[0][0] + sy2), R(P.win_min)), R(P.win_max));
        const R wz = std::min(std::max(R(P.win_nsigma) * std::sqrt(f.C[1][1] + sz2), R(P.win_min)), R(P.win_max));
        int32_t best = -1;
        R gb = 0, g2 = 0;
        bool have2 = false;
        for (int32_t c : rows[row]) {
            bool iy = le(std::fabs(R(gy[c]) - f.y), wy, mg);
            bool iz = le(std::fabs(R(gz[c]) - f.z), wz, mg);
            if (!(iy && iz)) continue;
            const R g = gate(f, R(gy[c]), R(gz[c]));
            if (best < 0 || g < gb) {
                if (best >= 0) { g2 = gb; have2 = true; }
                gb = g; best = c;
            } else if (!have2 || g < g2) { g2 = g; have2 = true; }
        }
        if (best < 0) return -1;
        if (have2) mg.rel((double)gb, (double)g2);
        return le(gb, R(P.chi2_ext), mg) ? best : -1;
    }

    /* ---- O5 tracklet constructor for the start hit h0 ---- */
    void construct(const Result& res, int32_t h0, Tracklet& T, std::vector<uint8_t>* used = nullptr, int32_t base = 0) const {
        Margin mg;
        std::vector<int32_t>& tab = T.table;
        tab.assign(n_rows, -1);
        const int r0 = grow[h0];
        const int32_t h1 = res.clink_up[h0];
        Fit<R> f, snap;
        {   /* initial state from the first link */
            const R dx = X[grow[h1]] - X[r0];
            const R dy = R(gy[h1]) - R(gy[h0]), dz = R(gz[h1]) - R(gz[h0]);
            const R dl = std::sqrt(dx * dx + dy * dy);
            f.y = R(gy[h0]); f.z = R(gz[h0]); f.s = dy / dl; f.t = dz / dl; f.q = R(0);
            prior(f); f.n = 1;
        }
        tab[r0] = h0;
        snap = f;
        int top = r0;
        /* up pass */
        {
            bool follow = true;
            int32_t cur = h1;
            int miss = 0;
            R xc = X[r0];
            for (int row = r0 + 1; row < n_rows; row++) {
                if (!transport(f, xc, X[row], mg)) break;
                xc = X[row];
                if (follow) {
                    if (row < grow[cur]) continue;
                    if (le(gate(f, R(gy[cur]), R(gz[cur])), R(P.chi2_link), mg)) {
                        update(f, cur); tab[row] = cur; snap = f; top = row;
                        cur = res.clink_up[cur];
                        if (cur < 0) follow = false;
                        continue;
                    }
                    follow = false; /* fall through: search this same row */
                }
                if (gt(std::fabs(f.y), X[row] * R(G.tan_half_angle) + R(P.edge_margin), mg)) break;
                const int32_t c = search(f, row, mg);
                if (c >= 0) { update(f, c); tab[row] = c; snap = f; top = row; miss = 0; }
                else if (++miss > P.max_gap) break;
            }
        }
        if (used)   /* seed de-duplication: the hits this up pass recorded (sector-local index = hit - base) */
            for (int row = r0; row <= top; row++) if (tab[row] >= 0) (*used)[tab[row] - base] = 1;
        /* down pass: fresh fit from the top recorded hit, direction and curvature from the up pass */
        int first = top;
        {
            const int32_t ht = tab[top];
            f.y = R(gy[ht]); f.z = R(gz[ht]); f.s = snap.s; f.t = snap.t; f.q = snap.q;
            prior(f); f.n = 1;
            snap = f;
            int miss = 0;
            R xc = X[top];
            int row = top - 1;
            for (; row >= 0; row--) {
                if (!transport(f, xc, X[row], mg)) break;
                xc = X[row];
                const int32_t hr = tab[row];
                if (hr >= 0) {
                    if (le(gate(f, R(gy[hr]), R(gz[hr])), R(P.chi2_link), mg)) { update(f, hr); snap = f; first = row; }
                    else tab[row] = -1;
                    continue;
                }
                const bool below = row < r0;
                if (below && gt(std::fabs(f.y), X[row] * R(G.tan_half_angle) + R(P.edge_margin), mg)) break;
                const int32_t c = search(f, row, mg);
                if (c >= 0) { update(f, c); tab[row] = c; snap = f; first = row; miss = 0; }
                else if (below && ++miss > P.max_gap) break;
            }
            for (; row >= 0; row--) tab[row] = -1; /* rows the pass never reached keep nothing */
        }
        T.first_row = first; T.last_row = top; T.n_hits = snap.n;
        T.par[0] = (double)snap.y; T.par[1] = (double)snap.z; T.par[2] = (double)snap.s;
        T.par[3] = (double)snap.t; T.par[4] = (double)snap.q;
        for (int i = 0; i < 5; i++) T.cov[i] = (double)snap.C[i][i];
        T.chi2 = (double)snap.chi2;
        T.margin = mg.m;
    }

    /* ---- O8 refit of a selected track over its final hit list ----
       hits: the track's hits, row-ascending (at most one per row).  No search and no gate: every hit of the list
       is a measurement.  Up pass from the lowest hit (direction from the first two hits, q = 0, prior covariance),
       transporting to every consecutive row; down pass = fresh fit at the top hit reached with (s, t, q) of the
       up pass.  A failed transport ends a pass.  Result = state after the last update of the down pass
       (x_ref = row of that hit), chi2 and hit count of the down pass.  Lists of fewer than 2 hits are left alone. */
    bool refit(const std::vector<int32_t>& hits, double par[5], double& chi2, int& n_fit, int& ref_row, double out[5],
               int& out_row) const {
        const int m = (int)hits.size();
        if (m < 2) return false;
        Margin mg;
        Fit<R> f, snap;
        const int32_t h0 = hits[0], h1 = hits[1];
        const int r0 = grow[h0];
        {
            const R dx = X[grow[h1]] - X[r0];
            const R dy = R(gy[h1]) - R(gy[h0]), dz = R(gz[h1]) - R(gz[h0]);
            const R dl = std::sqrt(dx * dx + dy * dy);
            f.y = R(gy[h0]); f.z = R(gz[h0]); f.s = dy / dl; f.t = dz / dl; f.q = R(0);
            prior(f); f.n = 1;
        }
        snap = f;
        int k_top = 0;                       /* position in the list of the last hit the up pass used */
        {
            R xc = X[r0];
            int k = 1;
            for (int row = r0 + 1; row <= grow[hits[m - 1]]; row++) {
                if (!transport(f, xc, X[row], mg)) break;
                xc = X[row];
                if (row == grow[hits[k]]) { update(f, hits[k]); snap = f; k_top = k; k++; }
            }
        }
        /* outer state: the up pass right after its last update (all hits below are in it) */
        out[0] = (double)snap.y; out[1] = (double)snap.z; out[2] = (double)snap.s; out[3] = (double)snap.t;
        out[4] = (double)snap.q; out_row = grow[hits[k_top]];
        {
            const int32_t ht = hits[k_top];
            f.y = R(gy[ht]); f.z = R(gz[ht]); f.s = snap.s; f.t = snap.t; f.q = snap.q;
            prior(f); f.n = 1;
            snap = f;
            ref_row = grow[ht];
            R xc = X[grow[ht]];
            int k = k_top - 1;
            for (int row = grow[ht] - 1; row >= r0; row--) {
                if (!transport(f, xc, X[row], mg)) break;
                xc = X[row];
                if (row == grow[hits[k]]) { update(f, hits[k]); snap = f; ref_row = row; k--; }
            }
        }
        par[0] = (double)snap.y; par[1] = (double)snap.z; par[2] = (double)snap.s; par[3] = (double)snap.t;
        par[4] = (double)snap.q;
        chi2 = (double)snap.chi2; n_fit = snap.n;
        return true;
    }
};


/* ---- O9 cross-sector merge ("merged together" PAPER.md:53) ----
 * Sectors: half = n_sectors / 2 per side, sector s = side * half + k, centre azimuth (k + 1/2) * 2 pi / half.
 * Segment A (sector s_A, outer state of its refit at pad row r_A) may continue in segment B of a sector next to it on
 * the same side whose first fitted row r_B obeys 1 <= r_B - r_A <= 1 + max_gap.  A's outer state is turned into
 * B's frame (angle alpha_A - alpha_B), moved along its helix to x = row_x[r_B] (state only, the O5 transport
 * formulas) and compared with B's parameters there:
 *   |dy| <= merge_dy, |dz| <= merge_dz, |d sin phi| <= merge_ds, |d tg lambda| <= merge_dt,
 *   D = (dy/merge_dy)^2 + (dz/merge_dz)^2 + (ds/merge_ds)^2 + (dt/merge_dt)^2.
 * next(A) = arg min_B D, prev(B) = arg min_A D (ties -> lowest track index); a link is kept when mutual. */
template <class R>
void merge_segments(const oracle_geometry& G, const oracle_params& P, Result& res) {
    const int T = (int)res.trk_sector.size();
    res.trk_next.assign(T, -1); res.trk_prev.assign(T, -1);
    res.trk_global.resize(T);
    for (int a = 0; a < T; a++) res.trk_global[a] = a;
    if (G.n_sectors < 4 || (G.n_sectors & 1)) return;
    const int half = G.n_sectors / 2;
    const double step = 2.0 * 3.14159265358979323846 / (double)half;
    const R cd = R(std::cos(step)), sd = R(std::sin(step));   /* rounded once to R */
    const R kB = R(-1) * (R(kLight) * R(G.bz));
    const R smax = R(P.sin_max);
    const R ty = R(P.merge_dy), tz = R(P.merge_dz), ts = R(P.merge_ds), tt = R(P.merge_dt);
    std::vector<R> bestn(T, R(0)), bestp(T, R(0));
    std::vector<Margin> mgs(T);
    res.trk_merge_margin.assign(T, std::numeric_limits<double>::infinity());
    /* mg: every float comparison of this pair leaves its relative margin there (parity protocol) */
    auto pair_score = [&](int a, int b, R& D, Margin& mg) -> bool {
        if (res.trk_row_out[a] < 0 || res.trk_row_out[b] < 0) return false;   /* no refit (fewer than 2 hits) */
        const int sa = res.trk_sector[a], sb = res.trk_sector[b];
        if (sa / half != sb / half) return false;
        const int dk = ((sb % half) - (sa % half) + half) % half;
        if (dk != 1 && dk != half - 1) return false;
        const int gap = res.trk_first_row[b] - res.trk_row_out[a];
        if (gap < 1 || gap > 1 + P.merge_max_gap) return false;
        const double* o = &res.trk_out[6 * (size_t)a];
        const R xa = R(o[0]), ya = R(o[1]), za = R(o[2]), s0 = R(o[3]), t0 = R(o[4]), q0 = R(o[5]);
        /* turn by alpha_A - alpha_B: -step when B is the next sector, +step when it is the one before */
        const R sn = (dk == 1) ? R(0) - sd : sd;
        if (gt(std::fabs(s0), smax, mg)) return false;
        const R c0a = std::sqrt(R(1) - s0 * s0);
        const R x1 = xa * cd - ya * sn;
        const R y1 = xa * sn + ya * cd;
        const R s1 = s0 * cd + c0a * sn;
        /* along the helix to B's reference row */
        const R xb = R(res.trk_x[b]);
        const R dx = xb - x1;
        const R kap = kB * q0;
        const R s2 = s1 + kap * dx;
        if (gt(std::fabs(s1), smax, mg)) return false;
        if (gt(std::fabs(s2), smax, mg)) return false;
        const R c1 = std::sqrt(R(1) - s1 * s1), c2 = std::sqrt(R(1) - s2 * s2);
        const R dy = dx * ((s1 + s2) * (R(1) / (c1 + c2)));
        const R dl2 = dx * dx + dy * dy;
        const R adl = std::sqrt(dl2);
        const R dl = (dx < R(0)) ? R(0) - adl : adl;
        const R u = kap * dl, u2 = u * u;
        const R dS = dl * (R(1) + u2 * (R(1) / R(24) + u2 * (R(3) / R(640))));
        const R y2 = y1 + dy, z2 = za + t0 * dS;
        const R ey = y2 - R(res.trk_y[b]), ez = z2 - R(res.trk_z[b]);
        const R es = s2 - R(res.trk_sinphi[b]), et = t0 - R(res.trk_tgl[b]);
        const bool iy = le(std::fabs(ey), ty, mg), iz = le(std::fabs(ez), tz, mg);
        const bool is = le(std::fabs(es), ts, mg), it = le(std::fabs(et), tt, mg);
        if (!(iy && iz && is && it)) return false;
        const R ny = ey * (R(1) / ty), nz = ez * (R(1) / tz), ns = es * (R(1) / ts), nt = et * (R(1) / tt);
        D = ((ny * ny + nz * nz) + ns * ns) + nt * nt;
        return true;
    };
    std::vector<int32_t> nx(T, -1), pv(T, -1);
    for (int a = 0; a < T; a++) {
        R second = 0; bool have2 = false;
        for (int b = 0; b < T; b++) {
            R D;
            if (a == b || !pair_score(a, b, D, mgs[a])) continue;
            if (nx[a] < 0 || D < bestn[a]) {                      /* ascending b: ties keep the lower index */
                if (nx[a] >= 0) { second = bestn[a]; have2 = true; }
                nx[a] = b; bestn[a] = D;
            } else if (!have2 || D < second) { second = D; have2 = true; }
        }
        if (have2) mgs[a].rel((double)bestn[a], (double)second);
    }
    for (int b = 0; b < T; b++) {
        R second = 0; bool have2 = false;
        for (int a = 0; a < T; a++) {
            R D;
            if (a == b || !pair_score(a, b, D, mgs[b])) continue;
            if (pv[b] < 0 || D < bestp[b]) {
                if (pv[b] >= 0) { second = bestp[b]; have2 = true; }
                pv[b] = a; bestp[b] = D;
            } else if (!have2 || D < second) { second = D; have2 = true; }
        }
        if (have2) mgs[b].rel((double)bestp[b], (double)second);
    }
    for (int a = 0; a < T; a++)
        if (nx[a] >= 0 && pv[nx[a]] == a) { res.trk_next[a] = nx[a]; res.trk_prev[nx[a]] = a; }
    for (int a = 0; a < T; a++) res.trk_merge_margin[a] = mgs[a].m;
    /* global track = chain of linked segments, named by its first segment (links join a sector to the next one
       outwards in row, so a chain cannot close on itself) */
    for (int a = 0; a < T; a++) {
        int h = a;
        while (res.trk_prev[h] >= 0) h = res.trk_prev[h];
        res.trk_global[a] = h;
    }
}

template <class R>
Result* run(const oracle_geometry& G, const oracle_params& P, int32_t n, const int32_t* sector_offset, const float* y,
            const float* z, const int32_t* row, int n_threads, int stop_after) {
    Result* res = new Result;
    res->n_clusters = n; res->n_sectors = G.n_sectors; res->n_rows = G.n_rows;
    res->link_up.assign(n, -1); res->link_dn.assign(n, -1);
    res->clink_up.assign(n, -1); res->clink_dn.assign(n, -1);
    res->nf_margin.assign(n, std::numeric_limits<double>::infinity());
    const int ns = G.n_sectors;
    std::vector<std::vector<int32_t>> seeds(ns);
    std::vector<std::vector<Tracklet>> tls(ns);
    /* per-sector output tracks */
    struct Refit { bool ok = false; double par[5] = {0, 0, 0, 0, 0}, chi2 = 0, out[5] = {0, 0, 0, 0, 0}; int n_fit = 0, ref_row = 0, out_row = -1; };
    struct Out { std::vector<int32_t> seed, nh, first_row; std::vector<std::vector<int32_t>> hits; std::vector<Refit> refit; };
    std::vector<Out> outs(ns);
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic, 1)
    for (int s = 0; s < ns; s++) {
        Sector<R> S(P, G, y, z, row);
        const int32_t b = sector_offset[s], e = sector_offset[s + 1];
        S.bucket(b, e);
        S.neighbours(*res);
        if (stop_after == 2) continue;
        S.clean(*res, b, e);
        S.start_hits(*res, seeds[s]);
        if (stop_after == 4) continue;
        tls[s].resize(seeds[s].size());
        {   /* O5 with seed de-duplication (R23): start hits are taken in canonical order (pad row, caller's
               index); every hit an up pass records is marked; a start hit that is already marked builds no tracklet
               (its track is being followed from below).  Marks come from up passes of lower rows only, so the
               order of the start hits inside a row plays no role. */
            std::vector<uint8_t> used(P.seed_dedup ? e - b : 0, 0);
            for (size_t i = 0; i < seeds[s].size(); i++) {
                if (P.seed_dedup && used[seeds[s][i] - b]) { tls[s][i].table.assign(G.n_rows, -1); continue; }
                S.construct(*res, seeds[s][i], tls[s][i], P.seed_dedup ? &used : nullptr, b);
            }
        }
        if (stop_after == 5) continue;
        /* ---- O6 selector ---- */
        /* owner(hit) = tracklet with most hits, ties -> lowest canonical id, among tracklets with
           n_hits >= min_tracklet_hits whose table contains the hit */
        std::vector<int32_t> owner(e - b, -1);
        for (size_t i = 0; i < tls[s].size(); i++) {
            const Tracklet& T = tls[s][i];
            if (T.n_hits < P.min_tracklet_hits) continue;
            for (int r = 0; r < G.n_rows; r++) {
                const int32_t h = T.table[r];
                if (h < 0) continue;
                int32_t& o = owner[h - b];
                if (o < 0 || T.n_hits > tls[s][o].n_hits) o = (int32_t)i; /* ascending i: ties keep the lower id */
            }
        }
        for (size_t i = 0; i < tls[s].size(); i++) {
            const Tracklet& T = tls[s][i];
            if (T.n_hits < P.min_tracklet_hits) continue;
            std::vector<int32_t> hits;
            for (int r = 0; r < G.n_rows; r++) {
                const int32_t h = T.table[r];
                if (h >= 0 && owner[h - b] == (int32_t)i) hits.push_back(h);
            }
            if ((int)hits.size() < P.min_track_hits) continue;
            outs[s].seed.push_back((int32_t)i);
            outs[s].nh.push_back((int32_t)hits.size());
            outs[s].first_row.push_back(T.first_row);
            Refit rf;   /* ---- O8 ---- */
            if (P.refit) rf.ok = S.refit(hits, rf.par, rf.chi2, rf.n_fit, rf.ref_row, rf.out, rf.out_row);
            outs[s].refit.push_back(rf);
            outs[s].hits.push_back(std::move(hits));
        }
    }
    /* ---- O7 output in canonical order (sector, start row, start-hit index) ---- */
    res->seed_offset.assign(ns + 1, 0);
    for (int s = 0; s < ns; s++) res->seed_offset[s + 1] = res->seed_offset[s] + (int32_t)seeds[s].size();
    for (int s = 0; s < ns; s++) {
        for (int32_t h : seeds[s]) res->start_hit.push_back(h);
        for (auto& T : tls[s]) res->tracklets.push_back(std::move(T));
    }
    for (int s = 0; s < ns; s++) {
        for (size_t k = 0; k < outs[s].seed.size(); k++) {
            const int32_t gid = res->seed_offset[s] + outs[s].seed[k];
            const Tracklet& T = res->tracklets[gid];
            res->trk_sector.push_back(s);
            res->trk_seed.push_back(gid);
            res->trk_first_hit.push_back((int32_t)res->hit_idx.size());
            res->trk_n_hits.push_back(outs[s].nh[k]);
            res->trk_ndf.push_back(2 * T.n_hits - 5);
            res->trk_first_row.push_back(T.first_row);
            res->trk_x.push_back((double)G.row_x[T.first_row]);
            res->trk_y.push_back(T.par[0]); res->trk_z.push_back(T.par[1]); res->trk_sinphi.push_back(T.par[2]);
            res->trk_tgl.push_back(T.par[3]); res->trk_qpt.push_back(T.par[4]);
            res->trk_chi2.push_back(T.chi2); res->trk_margin.push_back(T.margin);
            const Refit& rf = outs[s].refit[k];
            if (rf.ok) {   /* O8: parameters, chi2, ndf and reference row of the refit replace the tracklet's */
                res->trk_ndf.back() = 2 * rf.n_fit - 5;
                res->trk_first_row.back() = rf.ref_row;
                res->trk_x.back() = (double)G.row_x[rf.ref_row];
                res->trk_y.back() = rf.par[0]; res->trk_z.back() = rf.par[1]; res->trk_sinphi.back() = rf.par[2];
                res->trk_tgl.back() = rf.par[3]; res->trk_qpt.back() = rf.par[4]; res->trk_chi2.back() = rf.chi2;
            }
            res->trk_row_out.push_back(rf.ok ? rf.out_row : -1);
            res->trk_out.push_back(rf.ok ? (double)G.row_x[rf.out_row] : 0.0);
            for (int j = 0; j < 5; j++) res->trk_out.push_back(rf.ok ? rf.out[j] : 0.0);
            for (int32_t h : outs[s].hits[k]) res->hit_idx.push_back(h);
        }
    }
    {
        const size_t T = res->trk_sector.size();
        res->trk_g.assign(7 * T, 0.0); res->trk_g_ndf.assign(T, 0); res->trk_g_n_hits.assign(T, 0); res->trk_g_sector.assign(T, -1);
    }
    if (P.merge && P.refit && stop_after == 0) {
        merge_segments<R>(G, P, *res);
        /* ---- O10: one fit per global track ("global reconstruction") ---- */
        const int T = (int)res->trk_sector.size();
        const int half = G.n_sectors / 2;
        const double step = 2.0 * 3.14159265358979323846 / (double)std::max(half, 1);
        const R cd = R(std::cos(step)), sd = R(std::sin(step));
        Sector<R> S(P, G, y, z, row);
        std::vector<std::vector<int32_t>> hl(T);
        for (int a = 0; a < T; a++)
            hl[a].assign(res->hit_idx.begin() + res->trk_first_hit[a], res->hit_idx.begin() + res->trk_first_hit[a] + res->trk_n_hits[a]);
        for (int a = 0; a < T; a++) {
            if (res->trk_prev[a] >= 0 || res->trk_row_out[a] < 0) continue;   /* not the first segment / no refit */
            std::vector<const std::vector<int32_t>*> seg;
            std::vector<R> sn_up;
            for (int b = a, pb = -1; b >= 0; pb = b, b = res->trk_next[b]) {
                seg.push_back(&hl[b]);
                if (pb < 0) sn_up.push_back(R(0));
                else {
                    const int dk = ((res->trk_sector[b] % half) - (res->trk_sector[pb] % half) + half) % half;
                    sn_up.push_back(dk == 1 ? R(0) - sd : sd);
                }
            }
            double g[7];
            int n_fit = 0, end_seg = 0;
            if (!S.global_fit(seg, sn_up, cd, g, n_fit, end_seg)) continue;
            for (int j = 0; j < 7; j++) res->trk_g[7 * (size_t)a + j] = g[j];
            res->trk_g_ndf[a] = 2 * n_fit - 5; res->trk_g_n_hits[a] = n_fit;
            int b = a;
            for (int k = 0; k < end_seg; k++) b = res->trk_next[b];
            res->trk_g_sector[a] = res->trk_sector[b];
        }
    } else {
        const size_t T = res->trk_sector.size();
        res->trk_next.assign(T, -1); res->trk_prev.assign(T, -1); res->trk_global.resize(T);
        res->trk_merge_margin.assign(T, std::numeric_limits<double>::infinity());
        for (size_t a = 0; a < T; a++) res->trk_global[a] = (int32_t)a;
    }
    return res;
}

template <class T> void copy_out(const std::vector<T>& v, void* dst) {
    if (!v.empty()) std::memcpy(dst, v.data(), sizeof(T) * v.size());
}

} /* namespace */

extern "C" {

void oracle_default_params(oracle_params* p) {
    /* defaults of SURVEY.md 8(c).3 (validated by tests/test_oracle_e2e.py) */
    p->link_step = 1;
    p->nf_slope_y = 1.5f; p->nf_slope_z = 2.0f; p->nf_w0 = 0.3f; p->nf_dmax = 0.25f;
    p->sin_max = 0.95f;
    p->var_s = 0.25f; p->var_t = 1.0f; p->var_q = 100.0f;
    p->chi2_link = 25.0f; p->chi2_ext = 16.0f;
    p->win_nsigma = 4.0f; p->win_min = 0.3f; p->win_max = 3.0f;
    p->max_gap = 5; p->edge_margin = 1.0f;
    p->min_tracklet_hits = 10; p->min_track_hits = 10;
    p->refit = 0;
    p->merge = 0; p->merge_dy = 1.0f; p->merge_dz = 1.0f; p->merge_ds = 0.05f; p->merge_dt = 0.05f; p->merge_max_gap = 6;
    p->seed_dedup = 1;
    p->checked = 0;
}

/* precision: 0 = double, 1 = strict float32.  stop_after: 0 = everything, 2 = after O2, 4 = after O4,
 * 5 = after O5.  Returns an opaque result (oracle_free). */
void* oracle_track_event(const oracle_geometry* G, const oracle_params* P, int32_t precision, int32_t n_clusters,
                         const int32_t* sector_offset, const float* y, const float* z, const int32_t* row,
                         int32_t n_threads, int32_t stop_after) {
    if (!G || !P || !sector_offset || G->n_rows <= 0 || G->n_sectors <= 0) return nullptr;
    if (P->link_step < 1 || P->link_step > 2) return nullptr;
    for (int32_t i = 0; i < n_clusters; i++) {
        if (row[i] < 0 || row[i] >= G->n_rows) return nullptr;
        if (P->checked && !(std::isfinite(y[i]) && std::isfinite(z[i]))) return nullptr;
    }
    if (precision == 1) return run<float>(*G, *P, n_clusters, sector_offset, y, z, row, n_threads, stop_after);
    return run<double>(*G, *P, n_clusters, sector_offset, y, z, row, n_threads, stop_after);
}

void oracle_free(void* r) { delete static_cast<Result*>(r); }

/* sizes: [n_clusters, n_seeds, n_tracks, n_track_hits, n_rows] */
void oracle_sizes(const void* rv, int64_t* out) {
    const Result* r = static_cast<const Result*>(rv);
    out[0] = r->n_clusters; out[1] = (int64_t)r->start_hit.size(); out[2] = (int64_t)r->trk_sector.size();
    out[3] = (int64_t)r->hit_idx.size(); out[4] = r->n_rows;
}

enum {
    F_LINK_UP = 0, F_LINK_DN, F_CLINK_UP, F_CLINK_DN, F_NF_MARGIN, F_SEED_OFFSET, F_START_HIT,
    F_TL_FIRST_ROW, F_TL_LAST_ROW, F_TL_N_HITS, F_TL_PAR, F_TL_CHI2, F_TL_MARGIN, F_TL_TABLE,
    F_TRK_SECTOR, F_TRK_FIRST_HIT, F_TRK_N_HITS, F_TRK_NDF, F_TRK_SEED, F_TRK_FIRST_ROW,
    F_TRK_X, F_TRK_Y, F_TRK_Z, F_TRK_SINPHI, F_TRK_TGL, F_TRK_QPT, F_TRK_CHI2, F_TRK_MARGIN, F_HIT_IDX, F_TL_COV, F_TRK_ROW_OUT, F_TRK_OUT, F_TRK_NEXT, F_TRK_PREV, F_TRK_GLOBAL, F_TRK_MERGE_MARGIN,
    F_TRK_G, F_TRK_G_NDF, F_TRK_G_N_HITS, F_TRK_G_SECTOR
};

/* copy one result field into caller memory (int32 or float64, shapes in oracle/__init__.py) */
int32_t oracle_copy(const void* rv, int32_t field, void* dst) {
    const Result* r = static_cast<const Result*>(rv);
    const size_t S = r->tracklets.size();
    switch (field) {
        case F_LINK_UP: copy_out(r->link_up, dst); break;
        case F_LINK_DN: copy_out(r->link_dn, dst); break;
        case F_CLINK_UP: copy_out(r->clink_up, dst); break;
        case F_CLINK_DN: copy_out(r->clink_dn, dst); break;
        case F_NF_MARGIN: copy_out(r->nf_margin, dst); break;
        case F_SEED_OFFSET: copy_out(r->seed_offset, dst); break;
        case F_START_HIT: copy_out(r->start_hit, dst); break;
        case F_TL_FIRST_ROW: for (size_t i = 0; i < S; i++) ((int32_t*)dst)[i] = r->tracklets[i].first_row; break;
        case F_TL_LAST_ROW: for (size_t i = 0; i < S; i++) ((int32_t*)dst)[i] = r->tracklets[i].last_row; break;
        case F_TL_N_HITS: for (size_t i = 0; i < S; i++) ((int32_t*)dst)[i] = r->tracklets[i].n_hits; break;
        case F_TL_PAR: for (size_t i = 0; i < S; i++) std::memcpy((double*)dst + 5 * i, r->tracklets[i].par, 40); break;
        case F_TL_COV: for (size_t i = 0; i < S; i++) std::memcpy((double*)dst + 5 * i, r->tracklets[i].cov, 40); break;
        case F_TL_CHI2: for (size_t i = 0; i < S; i++) ((double*)dst)[i] = r->tracklets[i].chi2; break;
        case F_TL_MARGIN: for (size_t i = 0; i < S; i++) ((double*)dst)[i] = r->tracklets[i].margin; break;
        case F_TL_TABLE:
            for (size_t i = 0; i < S; i++)
                if (!r->tracklets[i].table.empty())
                    std::memcpy((int32_t*)dst + (size_t)r->n_rows * i, r->tracklets[i].table.data(), 4 * (size_t)r->n_rows);
            break;
        case F_TRK_SECTOR: copy_out(r->trk_sector, dst); break;
        case F_TRK_FIRST_HIT: copy_out(r->trk_first_hit, dst); break;
        case F_TRK_N_HITS: copy_out(r->trk_n_hits, dst); break;
        case F_TRK_NDF: copy_out(r->trk_ndf, dst); break;
        case F_TRK_SEED: copy_out(r->trk_seed, dst); break;
        case F_TRK_FIRST_ROW: copy_out(r->trk_first_row, dst); break;
        case F_TRK_X: copy_out(r->trk_x, dst); break;
        case F_TRK_Y: copy_out(r->trk_y, dst); break;
        case F_TRK_Z: copy_out(r->trk_z, dst); break;
        case F_TRK_SINPHI: copy_out(r->trk_sinphi, dst); break;
        case F_TRK_TGL: copy_out(r->trk_tgl, dst); break;
        case F_TRK_QPT: copy_out(r->trk_qpt, dst); break;
        case F_TRK_CHI2: copy_out(r->trk_chi2, dst); break;
        case F_TRK_MARGIN: copy_out(r->trk_margin, dst); break;
        case F_HIT_IDX: copy_out(r->hit_idx, dst); break;
        case F_TRK_ROW_OUT: copy_out(r->trk_row_out, dst); break;
        case F_TRK_OUT: copy_out(r->trk_out, dst); break;
        case F_TRK_NEXT: copy_out(r->trk_next, dst); break;
        case F_TRK_PREV: copy_out(r->trk_prev, dst); break;
        case F_TRK_GLOBAL: copy_out(r->trk_global, dst); break;
        case F_TRK_MERGE_MARGIN: copy_out(r->trk_merge_margin, dst); break;
        case F_TRK_G: copy_out(r->trk_g, dst); break;
        case F_TRK_G_NDF: copy_out(r->trk_g_ndf, dst); break;
        case F_TRK_G_N_HITS: copy_out(r->trk_g_n_hits, dst); break;
        case F_TRK_G_SECTOR: copy_out(r->trk_g_sector, dst); break;
        default: return -1;
    }
    return 0;
}

/* ---- single-step entry points for the pins (double and float) ---- */
/* state: [y z s t q], cov: 25 row-major.  Returns 0 ok, 1 transport failed. */
int32_t oracle_transport(const oracle_geometry* G, const oracle_params* P, int32_t precision, double x, double x1,
                         double* state, double* cov) {
    oracle_geometry g = *G;
    float rx[1] = {0.f};
    g.n_rows = 1; g.row_x = rx;
    Margin mg;
    if (precision == 1) {
        Sector<float> S(*P, g, nullptr, nullptr, nullptr);
        Fit<float> f;
        f.y = (float)state[0]; f.z = (float)state[1]; f.s = (float)state[2]; f.t = (float)state[3]; f.q = (float)state[4];
        for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) f.C[i][j] = (float)cov[5 * i + j];
        if (!S.transport(f, (float)x, (float)x1, mg)) return 1;
        state[0] = f.y; state[1] = f.z; state[2] = f.s; state[3] = f.t; state[4] = f.q;
        for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) cov[5 * i + j] = f.C[i][j];
    } else {
        Sector<double> S(*P, g, nullptr, nullptr, nullptr);
        Fit<double> f;
        f.y = state[0]; f.z = state[1]; f.s = state[2]; f.t = state[3]; f.q = state[4];
        for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) f.C[i][j] = cov[5 * i + j];
        if (!S.transport(f, x, x1, mg)) return 1;
        state[0] = f.y; state[1] = f.z; state[2] = f.s; state[3] = f.t; state[4] = f.q;
        for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) cov[5 * i + j] = f.C[i][j];
    }
    return 0;
}

/* one measurement update (y then z) in double; chi2 in/out */
void oracle_update(const oracle_geometry* G, const oracle_params* P, double my, double mz, double* state, double* cov,
                   double* chi2) {
    oracle_geometry g = *G;
    float rx[1] = {0.f};
    g.n_rows = 1; g.row_x = rx;
    Sector<double> S(*P, g, nullptr, nullptr, nullptr);
    Fit<double> f;
    f.y = state[0]; f.z = state[1]; f.s = state[2]; f.t = state[3]; f.q = state[4]; f.chi2 = *chi2; f.n = 0;
    for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) f.C[i][j] = cov[5 * i + j];
    S.update1(f, 0, my, (double)G->sigma_y * (double)G->sigma_y);
    S.update1(f, 1, mz, (double)G->sigma_z * (double)G->sigma_z);
    state[0] = f.y; state[1] = f.z; state[2] = f.s; state[3] = f.t; state[4] = f.q; *chi2 = f.chi2;
    for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) cov[5 * i + j] = f.C[i][j];
}

/* one rotation step of O10 in double: state [y z s t q], cov 25 row-major, x in/out; angle given by its sine / cosine.
 * Returns 0 ok, 1 failed. */
int32_t oracle_rotate(const oracle_geometry* G, const oracle_params* P, double* x, double sn, double cd, double* state,
                      double* cov) {
    oracle_geometry g = *G;
    float rx[1] = {0.f};
    g.n_rows = 1; g.row_x = rx;
    Margin mg;
    Sector<double> S(*P, g, nullptr, nullptr, nullptr);
    Fit<double> f;
    f.y = state[0]; f.z = state[1]; f.s = state[2]; f.t = state[3]; f.q = state[4];
    for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) f.C[i][j] = cov[5 * i + j];
    if (!S.rotate(f, *x, sn, cd, mg)) return 1;
    state[0] = f.y; state[1] = f.z; state[2] = f.s; state[3] = f.t; state[4] = f.q;
    for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) cov[5 * i + j] = f.C[i][j];
    return 0;
}

/* O9 on caller-given segments (for the pins): T segments with sector, first fitted row, parameters
 * par[T][6] = x y z sin phi tg lambda q/pT at that row, outer row and outer state out[T][6] (x y z s t q).
 * Fills next / prev / global [T] and margin [T] (may be NULL). */
int32_t oracle_merge_tracks(const oracle_geometry* G, const oracle_params* P, int32_t precision, int32_t T,
                            const int32_t* sector, const int32_t* first_row, const double* par, const int32_t* row_out,
                            const double* out, int32_t* next, int32_t* prev, int32_t* global, double* margin) {
    if (!G || !P || T < 0) return -1;
    Result res;
    res.n_sectors = G->n_sectors; res.n_rows = G->n_rows;
    for (int a = 0; a < T; a++) {
        res.trk_sector.push_back(sector[a]); res.trk_first_row.push_back(first_row[a]);
        res.trk_x.push_back(par[6 * a]); res.trk_y.push_back(par[6 * a + 1]); res.trk_z.push_back(par[6 * a + 2]);
        res.trk_sinphi.push_back(par[6 * a + 3]); res.trk_tgl.push_back(par[6 * a + 4]); res.trk_qpt.push_back(par[6 * a + 5]);
        res.trk_row_out.push_back(row_out[a]);
        for (int j = 0; j < 6; j++) res.trk_out.push_back(out[6 * a + j]);
    }
    if (precision == 1) merge_segments<float>(*G, *P, res); else merge_segments<double>(*G, *P, res);
    for (int a = 0; a < T; a++) {
        next[a] = res.trk_next[a]; prev[a] = res.trk_prev[a]; global[a] = res.trk_global[a];
        if (margin) margin[a] = res.trk_merge_margin.empty() ? std::numeric_limits<double>::infinity() : res.trk_merge_margin[a];
    }
    return 0;
}

int32_t oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

} /* extern "C" */
