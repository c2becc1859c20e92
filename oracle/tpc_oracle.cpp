/*
 * ORACLE — test infrastructure, NOT the product.
 *
 * Plain, slow, single-threaded C++17 implementation of Phase-I in-sector TPC tracking
 * (arxiv 1712.09430: seeding by cellular automaton, PAPER.md:33 / Fig. 3c; track following with a
 * simplified Kalman filter, PAPER.md:34,43 / Fig. 3d; tracklet selection), following
 * the readings S0..S6 and R-1..R-15 listed in DESIGN.md (the paper is an overview without
 * formulas; every numerical choice is a documented reading).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  It shares no code, header, table or constant with the CUDA
 * path under paper_1712_09430_b200/csrc.  The method is a heuristic plus an iteration, so the
 * oracle is the algorithm step by step in the order of DESIGN.md; the grid of S1 is an
 * accelerator only (brute_force=1 scans whole rows instead and must give identical results).
 *
 * Pins (tests/test_oracle_*.py): brute force == grid; analytic circle, group property and
 * finite-difference Jacobian of the propagation; closed-form least squares for the filter;
 * noise-free straight/helix recovery; pulls and chi2/ndf; chain/selector invariants; clean
 * single-track events found with all clusters; and for the control logic of constructTracklets /
 * roadSearch / selectTracklets (tests/test_oracle_legs.py): hand-counted gap bridging in legs B
 * and D (4 empty rows crossed, the 5th stops; counter from 0 at r0; leg C neither searches nor
 * counts), 9-vs-10 hits for kept tracklets and for owned hits, the road edge at
 * nsig*sqrt(C+err2) from the closed-form variance of a line fit, its cap and its rectangular
 * shape, the load-index tie-break of the search, and the restart of the inward pass against an
 * independent numpy filter.  No function here is "parity unpinned".
 *
 * Templated on the scalar type: double for the 1e-5 self-checks, float for GPU parity
 * (build with -O2 -ffp-contract=off: IEEE fp32; a fused multiply-add happens exactly where std::fma is written,
 * nowhere else; R-12).
 */
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

struct ParamsD {
    double err2_y, err2_z;       /* measurement variances */
    double nf_ty, nf_tz, nf_c;   /* neighbour window: |dy| <= nf_ty*|dx| + nf_c, |dz| <= nf_tz*|dx| + nf_c */
    double nf_d2max;             /* max squared collinearity residual of a triplet */
    double kf_css0, kf_ctt0, kf_ckk0; /* initial variances of sin(phi), dz/ds, q/pT */
    double kf_smax;              /* |sin(phi)| limit of the propagation */
    double road_nsig, road_max;  /* search road */
    int32_t max_gap, min_hits, seed_min_chain, pad;
    double merge_chi2;           /* S7: max chi2 (5 dof) of two matching track segments */
    int32_t merge_max_row_gap;   /* S7: max pad rows between the end of the inner and the start of the outer segment */
    int32_t pad2;
    double sector_dphi;          /* S7: angle between neighbouring sector frames [rad] */
    double field_ar, field_az;   /* S8: Bz(r, z) = Bz * (1 + field_ar * r^2 + field_az * z^2)  [1/cm^2] */
    double ms_x0_inv;            /* S8: 1 / radiation length of the gas [1/cm]; 0 = no multiple scattering */
};

/* ------------------------------------------------------------------ track model (S5) */
/* State at x: p = (y, z, s=sin(phi), t=dz/ds, k=q/pT); C symmetric 5x5 (full storage here). */
template <class T> struct State {
    T x;
    T p[5];
    T C[5][5];
    T chi2;
    int32_t nfit;
};

/* Propagation x -> x2, exact for a circle in a constant field, S5.
 * Returns false (state untouched) if |s| or |s2| >= smax.  J (optional) receives the Jacobian. */
template <class T> bool propagate(State<T> &st, T x2, T CB, T smax, T (*Jout)[5] = nullptr) {
    const T y = st.p[0], z = st.p[1], s = st.p[2], t = st.p[3], k = st.p[4];
    const T dx = x2 - st.x;
    const T kap = k * CB;
    const T s2 = std::fma(kap, dx, s);
    if (!(std::fabs(s) < smax) || !(std::fabs(s2) < smax)) return false;
    const T c = std::sqrt(std::fma(-s, s, T(1)));
    const T c2 = std::sqrt(std::fma(-s2, s2, T(1)));
    const T cc = c + c2;
    const T ss = s + s2;
    const T rcc = T(1) / cc;
    const T tg = ss * rcc;                      /* tan of the mean direction */
    const T q = std::sqrt(std::fma(tg, tg, T(1)));
    const T l = dx * q;                         /* signed chord */
    const T a = (T(0.5) * kap) * l;
    const T a2 = a * a;
    const T c16 = T(1) / T(6), c340 = T(3) / T(40);
    const T dS = l * std::fma(a2, std::fma(a2, c340, c16), T(1)); /* arc = chord * asin(a)/a, series */
    const T rc = T(1) / c, rc2 = T(1) / c2;
    const T rcc2 = rcc * rcc;
    const T d1 = std::fma(ss * s, rc, cc) * rcc2;   /* d tg / d s  */
    const T d2 = std::fma(ss * s2, rc2, cc) * rcc2; /* d tg / d s2 */
    T J[5][5];
    for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) J[i][j] = (i == j) ? T(1) : T(0);
    J[0][2] = dx * (d1 + d2);
    J[0][4] = ((dx * d2) * CB) * dx;
    J[2][4] = CB * dx;
    const T rq = T(1) / q;
    const T sm = tg * rq;                       /* = dy/l; d l / d tg = dx*sm, so d l / d s = sm*J[y][s] */
    const T tsm = t * sm;
    const T h = std::fma(a2, std::fma(a2, T(0.375), T(0.5)), T(1));   /* d dS / d l at fixed curvature */
    const T gp = std::fma(a2, T(3) / T(20), c16);                     /* d (dS/l) / d a2 */
    J[1][2] = (tsm * J[0][2]) * h;
    J[1][3] = dS;
    J[1][4] = std::fma(tsm * J[0][4], h, t * (((a * gp) * CB) * (l * l)));
    /* C2 = J C J^T: lower triangle, fused multiply-adds in ascending index order, then mirrored (no process noise) */
    T A[5][5];
    for (int i = 0; i < 5; i++)
        for (int j = 0; j < 5; j++) {
            T acc = T(0);
            for (int m = 0; m < 5; m++) acc = std::fma(J[i][m], st.C[m][j], acc);
            A[i][j] = acc;
        }
    T C2[5][5];
    for (int i = 0; i < 5; i++)
        for (int j = 0; j <= i; j++) {
            T acc = T(0);
            for (int m = 0; m < 5; m++) acc = std::fma(A[i][m], J[j][m], acc);
            C2[i][j] = acc;
            C2[j][i] = acc;
        }
    st.p[0] = std::fma(dx, tg, y);
    st.p[1] = std::fma(t, dS, z);
    st.p[2] = s2;
    st.x = x2;
    std::memcpy(st.C, C2, sizeof(C2));
    if (Jout) std::memcpy(Jout, J, sizeof(J));
    return true;
}

/* Textbook scalar Kalman update with measurement m of coordinate i (0=y, 1=z), variance e2. */
template <class T> void update1(State<T> &st, int i, T m, T e2) {
    const T r = m - st.p[i];
    const T S = st.C[i][i] + e2;
    const T w = T(1) / S;
    T K[5], row[5];
    for (int a = 0; a < 5; a++) { K[a] = st.C[a][i] * w; row[a] = st.C[i][a]; }
    for (int a = 0; a < 5; a++) st.p[a] = std::fma(K[a], r, st.p[a]);
    for (int a = 0; a < 5; a++)
        for (int b = 0; b <= a; b++) {
            const T v = std::fma(-K[a], row[b], st.C[a][b]);
            st.C[a][b] = v;
            st.C[b][a] = v;
        }
    st.chi2 = std::fma(r * r, w, st.chi2);
}

/* A hit = two sequential scalar updates, y first, then z (uncorrelated errors). */
template <class T> void update_hit(State<T> &st, T ym, T zm, T e2y, T e2z) {
    update1(st, 0, ym, e2y);
    update1(st, 1, zm, e2z);
    st.nfit++;
}

/* ------------------------------------------------------------------ Phase II: track merging (S7) */
/* Express the state in a frame rotated by +beta about z (x' = x cos b + y sin b, y' = -x sin b + y cos b), at the
 * plane x' = const through the state's own point.  cb, sb = cos/sin(beta) in working precision.  The track is assumed
 * to move towards +x in both frames (cos phi > 0); returns false (state untouched) if it does not in the new one or if
 * |sin phi'| >= smax.  Covariance: C' = J C J^T with the Jacobian of "rotate, then slide along the track back to
 * the plane" (S7): dy'/dy = c/c', dz'/dy = -t sb/c', ds'/dy = -k CB sb, ds'/ds = c'/c. */
template <class T> bool rotate(State<T> &st, T cb, T sb, T CB, T smax) {
    const T y = st.p[0], s = st.p[2], t = st.p[3], k = st.p[4];
    const T c = std::sqrt(T(1) - s * s);
    const T s2 = s * cb - c * sb;
    const T c2 = c * cb + s * sb;
    if (!(c2 > T(0)) || !(std::fabs(s2) < smax) || !(std::fabs(s) < smax)) return false;
    T J[5][5];
    for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) J[i][j] = (i == j) ? T(1) : T(0);
    J[0][0] = c / c2;
    J[1][0] = -(t * sb) / c2;
    J[2][0] = -((k * CB) * sb);
    J[2][2] = c2 / c;
    T A[5][5], C2[5][5];
    for (int i = 0; i < 5; i++)
        for (int j = 0; j < 5; j++) {
            T acc = T(0);
            for (int m = 0; m < 5; m++) acc = acc + J[i][m] * st.C[m][j];
            A[i][j] = acc;
        }
    for (int i = 0; i < 5; i++)
        for (int j = 0; j <= i; j++) {
            T acc = T(0);
            for (int m = 0; m < 5; m++) acc = acc + A[i][m] * J[j][m];
            C2[i][j] = acc; C2[j][i] = acc;
        }
    const T xn = st.x * cb + y * sb;
    st.p[0] = y * cb - st.x * sb;
    st.x = xn;
    st.p[2] = s2;
    std::memcpy(st.C, C2, sizeof(C2));
    return true;
}

/* chi2 = d^T S^-1 d for symmetric positive definite S (5x5), by LDL^T without pivoting; returns a huge value if a
 * pivot is not positive (then the two covariances carry no information and nothing is merged). */
template <class T> T chi2_5(const T d[5], const T S[5][5]) {
    T L[5][5], D[5];
    for (int j = 0; j < 5; j++) {
        T dj = S[j][j];
        for (int m = 0; m < j; m++) dj = dj - (L[j][m] * L[j][m]) * D[m];
        if (!(dj > T(0))) return T(1e30);
        D[j] = dj;
        for (int i = j + 1; i < 5; i++) {
            T v = S[i][j];
            for (int m = 0; m < j; m++) v = v - (L[i][m] * L[j][m]) * D[m];
            L[i][j] = v / dj;
        }
    }
    T w[5], chi = T(0);
    for (int i = 0; i < 5; i++) {               /* forward substitution L w = d, then sum w^2 / D */
        T v = d[i];
        for (int m = 0; m < i; m++) v = v - L[i][m] * w[m];
        w[i] = v;
        chi = chi + (v * v) / D[i];
    }
    return chi;
}

/* ------------------------------------------------------------------ the tracker */
struct TrackletOut {
    int64_t start_gid;
    int32_t sector, start_row, n_hits, first_row, last_row, kept, n_fit, near_tie;
    double x, p[5], c[15], chi2;
};
struct TrackOut {
    int64_t start_gid;
    int64_t cluster_offset;
    int32_t sector, n_clusters, first_row, last_row, n_fit, pad;
    double x, p[5], c[15], chi2;
};

template <class T> struct Tracker {
    int nSec, nRows;
    std::vector<T> rowX;
    ParamsD pd;
    T CB;
    /* params in working precision */
    T err2y, err2z, nfTy, nfTz, nfC, nfD2max, css0, ctt0, ckk0, smax, roadNsig, roadMax;

    std::vector<int64_t> rowBase;  /* [nSec*nRows+1] event-global id base of each (sector,row) */
    std::vector<T> y, z;
    int64_t N = 0;

    /* S1: per-row uniform grid (accelerator only) */
    struct Grid { T y0, z0, inv; int nY, nZ; std::vector<int32_t> start, idx; };
    std::vector<Grid> grid;
    static constexpr double kBin = 2.0;     /* cm */
    static constexpr double kMargin = 1e-3; /* cm, query slack; the exact window test follows */
    bool brute = false;

    std::vector<int32_t> linkUp, linkDn, linkUpC, linkDnC; /* row-local load index in row r+1 / r-1, -1 none */
    std::vector<uint8_t> tieS2;
    std::vector<int64_t> startHits;
    std::vector<TrackletOut> tracklets;
    std::vector<int32_t> rowHit;   /* [nTracklets*nRows] row-local load index, -1 none */
    std::vector<int64_t> owner;    /* [N] start_gid of the owning kept tracklet, -1 none */
    std::vector<TrackOut> tracks;
    std::vector<int32_t> clusterIds;
    double stageSec[6] = {0, 0, 0, 0, 0, 0};

    int cnt(int sr) const { return int(rowBase[sr + 1] - rowBase[sr]); }

    void buildGrid() {
        grid.assign(size_t(nSec) * nRows, Grid());
        for (int sr = 0; sr < nSec * nRows; sr++) {
            Grid &g = grid[sr];
            const int n = cnt(sr);
            const int64_t b = rowBase[sr];
            g.nY = g.nZ = 1; g.y0 = g.z0 = T(0); g.inv = T(1.0 / kBin);
            if (n == 0) { g.start.assign(2, 0); continue; }
            T ymin = y[b], ymax = y[b], zmin = z[b], zmax = z[b];
            for (int i = 1; i < n; i++) {
                ymin = std::min(ymin, y[b + i]); ymax = std::max(ymax, y[b + i]);
                zmin = std::min(zmin, z[b + i]); zmax = std::max(zmax, z[b + i]);
            }
            g.y0 = ymin; g.z0 = zmin;
            g.nY = std::max(1, std::min(4096, int(double(ymax - ymin) / kBin) + 1));
            g.nZ = std::max(1, std::min(4096, int(double(zmax - zmin) / kBin) + 1));
            g.start.assign(size_t(g.nY) * g.nZ + 1, 0);
            std::vector<int32_t> bin(n);
            for (int i = 0; i < n; i++) {
                bin[i] = binOf(g, z[b + i], g.z0, g.nZ) * g.nY + binOf(g, y[b + i], g.y0, g.nY);
                g.start[bin[i] + 1]++;
            }
            for (size_t k = 1; k < g.start.size(); k++) g.start[k] += g.start[k - 1];
            std::vector<int32_t> cur(g.start.begin(), g.start.end() - 1);
            g.idx.resize(n);
            for (int i = 0; i < n; i++) g.idx[cur[bin[i]]++] = i;
        }
    }
    static int binOf(const Grid &g, T v, T v0, int n) {
        double f = std::floor(double(v - v0) * double(g.inv));
        if (!(f > 0)) return 0;
        if (f > n - 1) return n - 1;
        return int(f);
    }
    /* enumerate every hit of row sr that can lie in [yc-wy, yc+wy] x [zc-wz, zc+wz] (superset) */
    template <class F> void forWindow(int sr, T yc, T zc, T wy, T wz, F &&f) const {
        const int n = cnt(sr);
        if (brute) { for (int i = 0; i < n; i++) f(i); return; }
        if (n == 0) return;
        const Grid &g = grid[sr];
        const T m = T(kMargin);
        const int by0 = binOf(g, yc - wy - m, g.y0, g.nY), by1 = binOf(g, yc + wy + m, g.y0, g.nY);
        const int bz0 = binOf(g, zc - wz - m, g.z0, g.nZ), bz1 = binOf(g, zc + wz + m, g.z0, g.nZ);
        for (int bz = bz0; bz <= bz1; bz++)
            for (int k = g.start[bz * g.nY + by0]; k < g.start[bz * g.nY + by1 + 1]; k++) f(g.idx[k]);
    }

    static bool nearRel(T a, T b) { return std::fabs(a - b) <= T(1e-6) * std::max(std::fabs(a), std::fabs(b)); }

    /* ---------------------------------------------------------------- S2 neighbours finder */
    void findNeighbours() {
        linkUp.assign(N, -1); linkDn.assign(N, -1); tieS2.assign(N, 0);
        std::vector<int32_t> U, D;
        for (int s = 0; s < nSec; s++)
            for (int r = 1; r <= nRows - 2; r++) {
                const int sr = s * nRows + r;
                const int n = cnt(sr);
                if (n == 0 || cnt(sr + 1) == 0 || cnt(sr - 1) == 0) continue;
                const T dxu = rowX[r + 1] - rowX[r];  /* > 0 */
                const T dxd = rowX[r - 1] - rowX[r];  /* < 0 */
                const T wu = -dxd / (dxu - dxd), wd = dxu / (dxu - dxd);
                const T wyU = nfTy * dxu + nfC, wzU = nfTz * dxu + nfC;
                const T wyD = nfTy * (-dxd) + nfC, wzD = nfTz * (-dxd) + nfC;
                const int64_t b = rowBase[sr], bu = rowBase[sr + 1], bd = rowBase[sr - 1];
                for (int h = 0; h < n; h++) {
                    const T yh = y[b + h], zh = z[b + h];
                    bool tie = false;
                    U.clear(); D.clear();
                    forWindow(sr + 1, yh, zh, wyU, wzU, [&](int i) {
                        const T ay = std::fabs(y[bu + i] - yh), az = std::fabs(z[bu + i] - zh);
                        if (ay <= wyU && az <= wzU) U.push_back(i);
                        if (nearRel(ay, wyU) || nearRel(az, wzU)) tie = true;
                    });
                    forWindow(sr - 1, yh, zh, wyD, wzD, [&](int i) {
                        const T ay = std::fabs(y[bd + i] - yh), az = std::fabs(z[bd + i] - zh);
                        if (ay <= wyD && az <= wzD) D.push_back(i);
                        if (nearRel(ay, wyD) || nearRel(az, wzD)) tie = true;
                    });
                    bool have = false; T best = T(0), second = T(-1); int bu_i = -1, bd_i = -1;
                    for (int u : U)
                        for (int d : D) {
                            const T ey = yh - (wu * y[bu + u] + wd * y[bd + d]);
                            const T ez = zh - (wu * z[bu + u] + wd * z[bd + d]);
                            const T d2 = ey * ey + ez * ez;
                            bool better = !have || d2 < best || (d2 == best && (u < bu_i || (u == bu_i && d < bd_i)));
                            if (better) { if (have) second = best; best = d2; bu_i = u; bd_i = d; have = true; }
                            else if (second < T(0) || d2 < second) second = d2;
                        }
                    if (have && second >= T(0) && nearRel(best, second)) tie = true;
                    if (have && nearRel(best, nfD2max)) tie = true;
                    if (have && best <= nfD2max) { linkUp[b + h] = bu_i; linkDn[b + h] = bd_i; }
                    tieS2[b + h] = tie ? 1 : 0;
                }
            }
    }

    /* ---------------------------------------------------------------- S3 neighbours cleaner */
    void cleanNeighbours() {
        linkUpC.assign(N, -1); linkDnC.assign(N, -1);
        for (int sr = 0; sr < nSec * nRows; sr++) {
            const int64_t b = rowBase[sr];
            for (int h = 0; h < cnt(sr); h++) {
                const int u = linkUp[b + h], d = linkDn[b + h];
                if (u >= 0 && linkDn[rowBase[sr + 1] + u] == h) linkUpC[b + h] = u;
                if (d >= 0 && linkUp[rowBase[sr - 1] + d] == h) linkDnC[b + h] = d;
            }
        }
    }

    /* ---------------------------------------------------------------- S4 start hits */
    void findStartHits() {
        startHits.clear();
        for (int sr = 0; sr < nSec * nRows; sr++) {
            const int64_t b = rowBase[sr];
            for (int h = 0; h < cnt(sr); h++) {
                if (linkDnC[b + h] >= 0) continue;
                /* chain of at least seed_min_chain hits above (and including) h */
                int len = 1, row = sr; int cur = h;
                while (len < pd.seed_min_chain) {
                    const int u = linkUpC[rowBase[row] + cur];
                    if (u < 0) break;
                    cur = u; row++; len++;
                }
                if (len >= pd.seed_min_chain) startHits.push_back(b + h);
            }
        }
    }

    /* ---------------------------------------------------------------- S5 tracklet constructor */
    void initCov(State<T> &st) const {
        for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) st.C[i][j] = T(0);
        st.C[0][0] = err2y; st.C[1][1] = err2z; st.C[2][2] = css0; st.C[3][3] = ctt0; st.C[4][4] = ckk0;
    }
    /* closest hit of row sr inside the covariance-sized road around the state; -1 if none */
    int roadSearch(int sr, const State<T> &st, bool &tie) const {
        T ry = roadNsig * std::sqrt(st.C[0][0] + err2y); if (!(ry < roadMax)) ry = roadMax;
        T rz = roadNsig * std::sqrt(st.C[1][1] + err2z); if (!(rz < roadMax)) rz = roadMax;
        const int64_t b = rowBase[sr];
        int best = -1; T bestD = T(0), second = T(-1);
        forWindow(sr, st.p[0], st.p[1], ry, rz, [&](int i) {
            const T dy = y[b + i] - st.p[0], dz = z[b + i] - st.p[1];
            const T ay = std::fabs(dy), az = std::fabs(dz);
            if (nearRel(ay, ry) || nearRel(az, rz)) tie = true;
            if (!(ay <= ry && az <= rz)) return;
            const T d = dy * dy + dz * dz;
            if (best < 0 || d < bestD || (d == bestD && i < best)) { if (best >= 0) second = bestD; bestD = d; best = i; }
            else if (second < T(0) || d < second) second = d;
        });
        if (best >= 0 && second >= T(0) && nearRel(bestD, second)) tie = true;
        return best;
    }

    void constructTracklets() {
        tracklets.clear(); rowHit.clear();
        std::vector<int32_t> rh(nRows);
        for (int64_t gid : startHits) {
            const int sr0 = int(std::upper_bound(rowBase.begin(), rowBase.end(), gid) - rowBase.begin()) - 1;
            const int s = sr0 / nRows, r0 = sr0 % nRows;
            const int h0 = int(gid - rowBase[sr0]);
            std::fill(rh.begin(), rh.end(), -1);
            bool tie = false;
            /* 1. init from the first link */
            const int h1 = linkUpC[gid];
            State<T> st;
            {
                const T dx = rowX[r0 + 1] - rowX[r0];
                const T dy = y[rowBase[sr0 + 1] + h1] - y[gid], dz = z[rowBase[sr0 + 1] + h1] - z[gid];
                const T l = std::sqrt(dx * dx + dy * dy);
                st.x = rowX[r0];
                st.p[0] = y[gid]; st.p[1] = z[gid]; st.p[2] = dy / l; st.p[3] = dz / l; st.p[4] = T(0);
                initCov(st); st.chi2 = T(0); st.nfit = 0;
            }
            rh[r0] = h0; int n = 1;
            int rTop = r0, hTop = h0; T sTop = st.p[2], tTop = st.p[3], kTop = st.p[4];
            /* 2. leg A: follow the cleaned links upward */
            int r = r0, cur = h0; bool alive = true;
            for (;;) {
                const int u = linkUpC[rowBase[s * nRows + r] + cur];
                if (u < 0) break;
                if (!propagate(st, rowX[r + 1], CB, smax)) { alive = false; break; }
                r++; cur = u;
                const int64_t g = rowBase[s * nRows + r] + u;
                update_hit(st, y[g], z[g], err2y, err2z);
                rh[r] = u; n++;
                rTop = r; hTop = u; sTop = st.p[2]; tTop = st.p[3]; kTop = st.p[4];
            }
            /* 3. leg B: extrapolate outward, closest hit in the road, at most max_gap empty rows in a row */
            if (alive) {
                int gap = 0;
                for (int rr = r + 1; rr < nRows; rr++) {
                    if (!propagate(st, rowX[rr], CB, smax)) break;
                    const int i = roadSearch(s * nRows + rr, st, tie);
                    if (i < 0) { if (++gap > pd.max_gap) break; continue; }
                    gap = 0;
                    const int64_t g = rowBase[s * nRows + rr] + i;
                    update_hit(st, y[g], z[g], err2y, err2z);
                    rh[rr] = i; n++;
                    rTop = rr; hTop = i; sTop = st.p[2]; tTop = st.p[3]; kTop = st.p[4];
                }
            }
            /* 4. leg C: re-initialise at the outermost hit, filter inward over all hits, extend below r0 */
            {
                const int64_t g = rowBase[s * nRows + rTop] + hTop;
                st.x = rowX[rTop];
                st.p[0] = y[g]; st.p[1] = z[g]; st.p[2] = sTop; st.p[3] = tTop; st.p[4] = kTop;
                initCov(st); st.chi2 = T(0); st.nfit = 0;
            }
            State<T> out = st;   /* output state = state after the last update of leg C */
            {
                int gap = 0;
                for (int rr = rTop - 1; rr >= 0; rr--) {
                    if (!propagate(st, rowX[rr], CB, smax)) break;
                    int i;
                    if (rr >= r0) { i = rh[rr]; if (i < 0) continue; }
                    else {
                        i = roadSearch(s * nRows + rr, st, tie);
                        if (i < 0) { if (++gap > pd.max_gap) break; continue; }
                        gap = 0; rh[rr] = i; n++;
                    }
                    const int64_t g = rowBase[s * nRows + rr] + i;
                    update_hit(st, y[g], z[g], err2y, err2z);
                    out = st;
                }
            }
            TrackletOut t; std::memset(&t, 0, sizeof(t));
            t.start_gid = gid; t.sector = s; t.start_row = r0; t.n_hits = n; t.near_tie = tie ? 1 : 0;
            t.first_row = -1; t.last_row = -1;
            for (int rr = 0; rr < nRows; rr++) if (rh[rr] >= 0) { if (t.first_row < 0) t.first_row = rr; t.last_row = rr; }
            t.kept = n >= pd.min_hits ? 1 : 0;          /* 5. */
            t.n_fit = out.nfit; t.x = double(out.x); t.chi2 = double(out.chi2);
            for (int i = 0; i < 5; i++) t.p[i] = double(out.p[i]);
            for (int i = 0, k = 0; i < 5; i++) for (int j = 0; j <= i; j++) t.c[k++] = double(out.C[i][j]);
            tracklets.push_back(t);
            rowHit.insert(rowHit.end(), rh.begin(), rh.end());
        }
    }

    /* ---------------------------------------------------------------- S6 tracklet selector */
    void selectTracklets() {
        owner.assign(N, -1);
        std::vector<int32_t> ownerN(N, 0);
        const size_t M = tracklets.size();
        for (size_t t = 0; t < M; t++) {
            const TrackletOut &tr = tracklets[t];
            if (!tr.kept) continue;
            for (int r = 0; r < nRows; r++) {
                const int i = rowHit[t * nRows + r];
                if (i < 0) continue;
                const int64_t g = rowBase[tr.sector * nRows + r] + i;
                /* best key: more hits, then smaller start-hit id */
                if (owner[g] < 0 || tr.n_hits > ownerN[g] || (tr.n_hits == ownerN[g] && tr.start_gid < owner[g])) {
                    owner[g] = tr.start_gid; ownerN[g] = tr.n_hits;
                }
            }
        }
        tracks.clear(); clusterIds.clear();
        for (size_t t = 0; t < M; t++) {
            const TrackletOut &tr = tracklets[t];
            if (!tr.kept) continue;
            std::vector<int32_t> ids; int first = -1, last = -1;
            for (int r = 0; r < nRows; r++) {
                const int i = rowHit[t * nRows + r];
                if (i < 0) continue;
                const int64_t g = rowBase[tr.sector * nRows + r] + i;
                if (owner[g] != tr.start_gid) continue;
                ids.push_back(int32_t(g)); if (first < 0) first = r; last = r;
            }
            if (int(ids.size()) < pd.min_hits) continue;
            TrackOut o; std::memset(&o, 0, sizeof(o));
            o.start_gid = tr.start_gid; o.cluster_offset = int64_t(clusterIds.size());
            o.sector = tr.sector; o.n_clusters = int32_t(ids.size()); o.first_row = first; o.last_row = last;
            o.n_fit = tr.n_fit; o.x = tr.x; o.chi2 = tr.chi2;
            std::memcpy(o.p, tr.p, sizeof(o.p)); std::memcpy(o.c, tr.c, sizeof(o.c));
            tracks.push_back(o);
            clusterIds.insert(clusterIds.end(), ids.begin(), ids.end());
        }
    }

    /* ---------------------------------------------------------------- S7 track merging (Phase II) */
    /* Per Phase-I track i (index into tracks): the segment that continues it outward / inward, -1 none. */
    std::vector<int32_t> mergeNext, mergePrev;
    std::vector<double> mergeChi2;          /* chi2 of the link i -> mergeNext[i] */
    std::vector<uint8_t> mergeTie;          /* the decision for track i was within 1e-6 relative of another one */
    std::vector<int32_t> mergedOffset, mergedSegs;   /* merged tracks: segments of merged track m = mergedSegs[off[m]..off[m+1]) */

    /* chi2 between segment a (inner) and segment b (outer): a's state is brought into b's sector frame and to b's
     * reference x (rotate, then propagate), then compared with b's state using the sum of the covariances.  < 0: no
     * match possible (different side, not neighbouring sectors, wrong order in rows, propagation fails). */
    T pairChi2(const TrackOut &a, const TrackOut &b) const {
        const int perSide = nSec >= 36 ? 18 : nSec;          /* sectors per TPC half (fewer in small test geometries) */
        if (a.sector / perSide != b.sector / perSide) return T(-1);
        const int sa = a.sector % perSide, sb_ = b.sector % perSide;
        int dsec = sb_ - sa;                                  /* -1, 0, +1 modulo the ring */
        if (dsec > perSide / 2) dsec -= perSide;
        if (dsec < -perSide / 2) dsec += perSide;
        if (dsec < -1 || dsec > 1) return T(-1);
        if (!(b.first_row > a.last_row) || b.first_row - a.last_row > pd.merge_max_row_gap) return T(-1);
        State<T> st;
        st.x = T(a.x); st.chi2 = T(0); st.nfit = 0;
        for (int i = 0; i < 5; i++) st.p[i] = T(a.p[i]);
        for (int i = 0, k = 0; i < 5; i++) for (int j = 0; j <= i; j++) { st.C[i][j] = st.C[j][i] = T(a.c[k++]); }
        if (dsec != 0) {
            const double beta = double(dsec) * pd.sector_dphi;       /* b's frame is a's rotated by +beta */
            if (!rotate(st, T(std::cos(beta)), T(std::sin(beta)), CB, smax)) return T(-1);
        }
        if (!propagate(st, T(b.x), CB, smax)) return T(-1);
        T d[5], S[5][5];
        for (int i = 0; i < 5; i++) d[i] = st.p[i] - T(b.p[i]);
        for (int i = 0, k = 0; i < 5; i++) for (int j = 0; j <= i; j++) { const T v = st.C[i][j] + T(b.c[k++]); S[i][j] = v; S[j][i] = v; }
        return chi2_5(d, S);
    }

    void mergeTracks() {
        const int n = int(tracks.size());
        mergeNext.assign(n, -1); mergePrev.assign(n, -1); mergeChi2.assign(n, 0.0); mergeTie.assign(n, 0);
        std::vector<T> bestOut(n, T(0)), bestIn(n, T(0));
        std::vector<int32_t> out(n, -1), in(n, -1);
        const T cut = T(pd.merge_chi2);
        /* canonical key of a track = id of its first cluster */
        auto key = [&](int i) { return clusterIds[tracks[i].cluster_offset]; };
        for (int a = 0; a < n; a++)
            for (int b = 0; b < n; b++) {
                if (a == b) continue;
                const T c = pairChi2(tracks[a], tracks[b]);
                if (c < T(0)) continue;
                if (nearRel(c, cut)) { mergeTie[a] = 1; mergeTie[b] = 1; }
                if (!(c <= cut)) continue;
                /* best outer partner of a, best inner partner of b: smaller chi2, then smaller key */
                if (out[a] >= 0 && nearRel(c, bestOut[a])) mergeTie[a] = 1;
                if (out[a] < 0 || c < bestOut[a] || (c == bestOut[a] && key(b) < key(out[a]))) { out[a] = b; bestOut[a] = c; }
                if (in[b] >= 0 && nearRel(c, bestIn[b])) mergeTie[b] = 1;
                if (in[b] < 0 || c < bestIn[b] || (c == bestIn[b] && key(a) < key(in[b]))) { in[b] = a; bestIn[b] = c; }
            }
        /* a link survives if it is mutual (as in the neighbours cleaner, S3) */
        for (int a = 0; a < n; a++)
            if (out[a] >= 0 && in[out[a]] == a) { mergeNext[a] = out[a]; mergePrev[out[a]] = a; mergeChi2[a] = double(bestOut[a]); }
        /* merged tracks: chains from the segments without an inner partner, in ascending key of that segment */
        std::vector<int> heads;
        for (int i = 0; i < n; i++) if (mergePrev[i] < 0) heads.push_back(i);
        std::sort(heads.begin(), heads.end(), [&](int x, int y) { return key(x) < key(y); });
        mergedOffset.assign(1, 0); mergedSegs.clear();
        for (int h : heads) {
            for (int i = h; i >= 0; i = mergeNext[i]) mergedSegs.push_back(i);
            mergedOffset.push_back(int32_t(mergedSegs.size()));
        }
    }

    /* ---------------------------------------------------------------- S8 final fit of the merged tracks (Phase II) */
    /* "the full track is refit using the full Kalman filter.  A polynomial approximation of the magnetic
     * field avoids the slow memory access to a field map."  Reading R-17 (S8): one inward filter pass over ALL
     * clusters of a merged track, from its outermost cluster to its innermost one, across the sector frames of its
     * segments; per step the field is the polynomial evaluated at the state's point, and multiple scattering over the
     * step's path is added to the covariance. */
    struct RefitOut { int32_t first_track, sector, n_fit, ok; double x, p[5], c[15], chi2; };
    std::vector<RefitOut> refits;           /* one per merged track, in the order of mergedOffset */

    int rowOfCluster(int64_t g) const {
        const int sr = int(std::upper_bound(rowBase.begin(), rowBase.end(), g) - rowBase.begin()) - 1;
        return sr % nRows;
    }
    T fieldCB(const State<T> &st) const {   /* curvature constant with the field at the state's point */
        const T r2 = st.x * st.x + st.p[0] * st.p[0];
        return CB * (T(1) + T(pd.field_ar) * r2 + T(pd.field_az) * (st.p[1] * st.p[1]));
    }
    /* multiple scattering over a straight path of length L (Highland without the log term, beta = 1):
     * theta0^2 = (0.0136 GeV / p)^2 L / X0, 1/p = |k| / sqrt(1 + t^2); projected on (sin phi, dz/ds, q/pT) */
    void addScattering(State<T> &st, T L) const {
        if (!(pd.ms_x0_inv > 0.0)) return;
        const T s = st.p[2], t = st.p[3], k = st.p[4];
        const T one_t2 = T(1) + t * t;
        const T th2 = (T(0.0136) * T(0.0136)) * ((k * k) / one_t2) * (L * T(pd.ms_x0_inv));
        st.C[2][2] = st.C[2][2] + (th2 * (T(1) - s * s)) * one_t2;
        st.C[3][3] = st.C[3][3] + (th2 * one_t2) * one_t2;
        const T c43 = ((th2 * t) * k) * one_t2;
        st.C[4][3] = st.C[4][3] + c43; st.C[3][4] = st.C[4][3];
        st.C[4][4] = st.C[4][4] + ((th2 * t) * t) * (k * k);
    }

    void refitMerged() {
        refits.clear();
        const int perSide = nSec >= 36 ? 18 : nSec;
        for (size_t m = 0; m + 1 < mergedOffset.size(); m++) {
            const int s0 = mergedOffset[m], s1 = mergedOffset[m + 1];
            const TrackOut &inner = tracks[mergedSegs[s0]];
            RefitOut o; std::memset(&o, 0, sizeof(o));
            o.first_track = mergedSegs[s0]; o.sector = inner.sector;
            /* default output: the innermost segment's Phase-I state (kept if the refit cannot be done) */
            o.x = inner.x; o.chi2 = inner.chi2; o.n_fit = 0; o.ok = 0;
            std::memcpy(o.p, inner.p, sizeof(o.p)); std::memcpy(o.c, inner.c, sizeof(o.c));
            /* start: the outermost segment's state taken to the pad row of its outermost cluster */
            const TrackOut &outer = tracks[mergedSegs[s1 - 1]];
            State<T> st; st.x = T(outer.x); st.chi2 = T(0); st.nfit = 0;
            for (int i = 0; i < 5; i++) st.p[i] = T(outer.p[i]);
            for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) st.C[i][j] = T(0);
            bool ok = propagate(st, rowX[outer.last_row], fieldCB(st), smax);
            int curSector = outer.sector;
            bool first = true;
            for (int sg = s1 - 1; ok && sg >= s0; sg--) {
                const TrackOut &seg = tracks[mergedSegs[sg]];
                for (int c = seg.n_clusters - 1; ok && c >= 0; c--) {
                    const int64_t g = clusterIds[seg.cluster_offset + c];
                    const int row = rowOfCluster(g);
                    if (first) {           /* the outermost cluster is the starting point, not a measurement */
                        st.p[0] = y[g]; st.p[1] = z[g]; st.x = rowX[row];
                        initCov(st); st.chi2 = T(0); st.nfit = 0;
                        first = false;
                        continue;
                    }
                    if (seg.sector != curSector) {   /* into the next segment's sector frame (S7 rotation) */
                        int dsec = seg.sector % perSide - curSector % perSide;
                        if (dsec > perSide / 2) dsec -= perSide;
                        if (dsec < -perSide / 2) dsec += perSide;
                        const double beta = double(dsec) * pd.sector_dphi;
                        ok = rotate(st, T(std::cos(beta)), T(std::sin(beta)), fieldCB(st), smax);
                        curSector = seg.sector;
                        if (!ok) break;
                    }
                    const T x0 = st.x, y0 = st.p[0], z0 = st.p[1];
                    ok = propagate(st, rowX[row], fieldCB(st), smax);
                    if (!ok) break;
                    const T dx = st.x - x0, dy = st.p[0] - y0, dz = st.p[1] - z0;
                    addScattering(st, std::sqrt((dx * dx + dy * dy) + dz * dz));
                    update_hit(st, y[g], z[g], err2y, err2z);
                }
            }
            if (ok && !first) {
                o.ok = 1; o.x = double(st.x); o.chi2 = double(st.chi2); o.n_fit = st.nfit; o.sector = curSector;
                for (int i = 0; i < 5; i++) o.p[i] = double(st.p[i]);
                for (int i = 0, k = 0; i < 5; i++) for (int j = 0; j <= i; j++) o.c[k++] = double(st.C[i][j]);
            }
            refits.push_back(o);
        }
    }

    void run(const int32_t *rowCounts, const float *yin, const float *zin, int bruteForce) {
        using clk = std::chrono::steady_clock;
        brute = bruteForce != 0;
        const int nsr = nSec * nRows;
        rowBase.assign(nsr + 1, 0);
        for (int i = 0; i < nsr; i++) rowBase[i + 1] = rowBase[i] + rowCounts[i];
        N = rowBase[nsr];
        y.resize(N); z.resize(N);
        for (int64_t i = 0; i < N; i++) { y[i] = T(yin[i]); z[i] = T(zin[i]); }
        auto t0 = clk::now();
        if (!brute) buildGrid();
        auto t1 = clk::now(); findNeighbours();
        auto t2 = clk::now(); cleanNeighbours();
        auto t3 = clk::now(); findStartHits();
        auto t4 = clk::now(); constructTracklets();
        auto t5 = clk::now(); selectTracklets();
        auto t6 = clk::now();
        auto sec = [](clk::time_point a, clk::time_point b) { return std::chrono::duration<double>(b - a).count(); };
        stageSec[0] = sec(t0, t1); stageSec[1] = sec(t1, t2); stageSec[2] = sec(t2, t3);
        stageSec[3] = sec(t3, t4); stageSec[4] = sec(t4, t5); stageSec[5] = sec(t5, t6);
    }

    Tracker(int ns, int nr, const float *rx, double bz, const ParamsD &p) : nSec(ns), nRows(nr), pd(p) {
        rowX.resize(nr);
        for (int i = 0; i < nr; i++) rowX[i] = T(rx[i]);
        CB = T(-0.299792458e-2 * bz);   /* curvature per unit q/pT [1/cm per c/GeV], constant field */
        err2y = T(p.err2_y); err2z = T(p.err2_z); nfTy = T(p.nf_ty); nfTz = T(p.nf_tz); nfC = T(p.nf_c);
        nfD2max = T(p.nf_d2max); css0 = T(p.kf_css0); ctt0 = T(p.kf_ctt0); ckk0 = T(p.kf_ckk0);
        smax = T(p.kf_smax); roadNsig = T(p.road_nsig); roadMax = T(p.road_max);
    }
};

struct Handle {
    int useDouble;
    Tracker<float> *f = nullptr;
    Tracker<double> *d = nullptr;
};


}  // namespace

/* ---- primitives exposed for the pins (tests/test_oracle_kalman.py) ---- */
/* state in/out: x[1], p[5], c[15] lower triangle (yy, zy,zz, sy,sz,ss, ty,tz,ts,tt, ky,kz,ks,kt,kk); J out 25 (may be null) */
template <class T> static int propagate_c(double *x, double *p, double *c, double x2, double CB, double smax, double *J) {
    State<T> st; st.x = T(*x); st.chi2 = T(0); st.nfit = 0;
    for (int i = 0; i < 5; i++) st.p[i] = T(p[i]);
    for (int i = 0, k = 0; i < 5; i++) for (int j = 0; j <= i; j++) { st.C[i][j] = st.C[j][i] = T(c[k++]); }
    T Jm[5][5];
    if (!propagate(st, T(x2), T(CB), T(smax), Jm)) return 0;
    *x = double(st.x);
    for (int i = 0; i < 5; i++) p[i] = double(st.p[i]);
    for (int i = 0, k = 0; i < 5; i++) for (int j = 0; j <= i; j++) c[k++] = double(st.C[i][j]);
    if (J) for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) J[i * 5 + j] = double(Jm[i][j]);
    return 1;
}
template <class T> static void update_c(double *p, double *c, double *chi2, int coord, double m, double e2) {
    State<T> st; st.x = T(0); st.chi2 = T(*chi2); st.nfit = 0;
    for (int i = 0; i < 5; i++) st.p[i] = T(p[i]);
    for (int i = 0, k = 0; i < 5; i++) for (int j = 0; j <= i; j++) { st.C[i][j] = st.C[j][i] = T(c[k++]); }
    update1(st, coord, T(m), T(e2));
    for (int i = 0; i < 5; i++) p[i] = double(st.p[i]);
    for (int i = 0, k = 0; i < 5; i++) for (int j = 0; j <= i; j++) c[k++] = double(st.C[i][j]);
    *chi2 = double(st.chi2);
}

#define DISPATCH(h, expr) ((h)->useDouble ? ((h)->d->expr) : ((h)->f->expr))

/* memcpy for the getters: an empty std::vector may hand out a null data() pointer, which memcpy must not be given */
static inline void copy_out(void *dst, const void *src, size_t bytes) { if (bytes) std::memcpy(dst, src, bytes); }
extern "C" {

void oracle_default_params(ParamsD *p) {
    p->err2_y = 0.01; p->err2_z = 0.01;
    p->nf_ty = 1.0; p->nf_tz = 1.5; p->nf_c = 0.5; p->nf_d2max = 0.25;
    p->kf_css0 = 1.0; p->kf_ctt0 = 10.0; p->kf_ckk0 = 100.0; p->kf_smax = 0.95;
    p->road_nsig = 4.0; p->road_max = 2.0;
    p->max_gap = 4; p->min_hits = 10; p->seed_min_chain = 3; p->pad = 0;
    p->merge_chi2 = 50.0; p->merge_max_row_gap = 40; p->pad2 = 0;
    p->sector_dphi = 20.0 * 3.14159265358979323846 / 180.0;
    p->field_ar = 0.0; p->field_az = 0.0; p->ms_x0_inv = 0.0;
}

void *oracle_create(int n_sectors, int n_rows, const float *row_x, double bz, const ParamsD *p, int use_double) {
    ParamsD d;
    if (p) d = *p; else oracle_default_params(&d);
    Handle *h = new Handle();
    h->useDouble = use_double;
    if (use_double) h->d = new Tracker<double>(n_sectors, n_rows, row_x, bz, d);
    else h->f = new Tracker<float>(n_sectors, n_rows, row_x, bz, d);
    return h;
}
void oracle_destroy(void *hv) { Handle *h = (Handle *)hv; if (!h) return; delete h->f; delete h->d; delete h; }

void oracle_run(void *hv, const int32_t *row_counts, const float *y, const float *z, int brute_force) {
    Handle *h = (Handle *)hv;
    if (h->useDouble) h->d->run(row_counts, y, z, brute_force); else h->f->run(row_counts, y, z, brute_force);
}
int64_t oracle_n_clusters(void *hv) { Handle *h = (Handle *)hv; return DISPATCH(h, N); }
/* which: 0 linkUp raw, 1 linkDn raw, 2 linkUp cleaned, 3 linkDn cleaned */
void oracle_get_links(void *hv, int which, int32_t *dst) {
    Handle *h = (Handle *)hv;
    auto cp = [&](auto &t) {
        const std::vector<int32_t> *v = which == 0 ? &t.linkUp : which == 1 ? &t.linkDn : which == 2 ? &t.linkUpC : &t.linkDnC;
        copy_out(dst, v->data(), v->size() * sizeof(int32_t));
    };
    if (h->useDouble) cp(*h->d); else cp(*h->f);
}
void oracle_get_tie_flags(void *hv, uint8_t *dst) {
    Handle *h = (Handle *)hv;
    if (h->useDouble) copy_out(dst, h->d->tieS2.data(), h->d->tieS2.size());
    else copy_out(dst, h->f->tieS2.data(), h->f->tieS2.size());
}
int64_t oracle_n_start_hits(void *hv) { Handle *h = (Handle *)hv; return (int64_t)DISPATCH(h, startHits.size()); }
void oracle_get_start_hits(void *hv, int64_t *dst) {
    Handle *h = (Handle *)hv;
    if (h->useDouble) copy_out(dst, h->d->startHits.data(), h->d->startHits.size() * 8);
    else copy_out(dst, h->f->startHits.data(), h->f->startHits.size() * 8);
}
int64_t oracle_n_tracklets(void *hv) { Handle *h = (Handle *)hv; return (int64_t)DISPATCH(h, tracklets.size()); }
int32_t oracle_sizeof_tracklet(void) { return (int32_t)sizeof(TrackletOut); }
int32_t oracle_sizeof_track(void) { return (int32_t)sizeof(TrackOut); }
void oracle_get_tracklets(void *hv, void *dst, int32_t *row_hit) {
    Handle *h = (Handle *)hv;
    auto cp = [&](auto &t) {
        copy_out(dst, t.tracklets.data(), t.tracklets.size() * sizeof(TrackletOut));
        copy_out(row_hit, t.rowHit.data(), t.rowHit.size() * sizeof(int32_t));
    };
    if (h->useDouble) cp(*h->d); else cp(*h->f);
}
void oracle_get_owners(void *hv, int64_t *dst) {
    Handle *h = (Handle *)hv;
    if (h->useDouble) copy_out(dst, h->d->owner.data(), h->d->owner.size() * 8);
    else copy_out(dst, h->f->owner.data(), h->f->owner.size() * 8);
}
int64_t oracle_n_tracks(void *hv) { Handle *h = (Handle *)hv; return (int64_t)DISPATCH(h, tracks.size()); }
int64_t oracle_n_cluster_ids(void *hv) { Handle *h = (Handle *)hv; return (int64_t)DISPATCH(h, clusterIds.size()); }
void oracle_get_tracks(void *hv, void *dst, int32_t *cluster_ids) {
    Handle *h = (Handle *)hv;
    auto cp = [&](auto &t) {
        copy_out(dst, t.tracks.data(), t.tracks.size() * sizeof(TrackOut));
        copy_out(cluster_ids, t.clusterIds.data(), t.clusterIds.size() * sizeof(int32_t));
    };
    if (h->useDouble) cp(*h->d); else cp(*h->f);
}
void oracle_get_stage_seconds(void *hv, double *dst) {
    Handle *h = (Handle *)hv;
    copy_out(dst, h->useDouble ? h->d->stageSec : h->f->stageSec, 6 * sizeof(double));
}

/* ---- Phase II (S7): run after oracle_run; results indexed like the tracks of oracle_get_tracks ---- */
void oracle_merge(void *hv) { Handle *h = (Handle *)hv; if (h->useDouble) h->d->mergeTracks(); else h->f->mergeTracks(); }
int64_t oracle_n_merged(void *hv) { Handle *h = (Handle *)hv; return (int64_t)DISPATCH(h, mergedOffset.size()) - 1; }
void oracle_get_merge(void *hv, int32_t *next, int32_t *prev, double *chi2, uint8_t *tie, int32_t *merged_offset, int32_t *merged_segs) {
    Handle *h = (Handle *)hv;
    auto cp = [&](auto &t) {
        const size_t n = t.mergeNext.size();
        copy_out(next, t.mergeNext.data(), n * 4); copy_out(prev, t.mergePrev.data(), n * 4);
        copy_out(chi2, t.mergeChi2.data(), n * 8); copy_out(tie, t.mergeTie.data(), n);
        copy_out(merged_offset, t.mergedOffset.data(), t.mergedOffset.size() * 4);
        copy_out(merged_segs, t.mergedSegs.data(), t.mergedSegs.size() * 4);
    };
    if (h->useDouble) cp(*h->d); else cp(*h->f);
}
/* primitive for the pins: covariance after multiple scattering over a path L [cm] in a gas of radiation length 1/x0_inv */
void oracle_scatter(const double *p, double *c, double L, double x0_inv) {
    ParamsD pd; oracle_default_params(&pd); pd.ms_x0_inv = x0_inv;
    const float rx[3] = {1.f, 2.f, 3.f};
    Tracker<double> t(1, 3, rx, 0.5, pd);
    State<double> st; st.x = 0; st.chi2 = 0; st.nfit = 0;
    for (int i = 0; i < 5; i++) st.p[i] = p[i];
    for (int i = 0, k = 0; i < 5; i++) for (int j = 0; j <= i; j++) { st.C[i][j] = st.C[j][i] = c[k++]; }
    t.addScattering(st, L);
    for (int i = 0, k = 0; i < 5; i++) for (int j = 0; j <= i; j++) c[k++] = st.C[i][j];
}
void oracle_refit(void *hv) { Handle *h = (Handle *)hv; if (h->useDouble) h->d->refitMerged(); else h->f->refitMerged(); }
int32_t oracle_sizeof_refit(void) { return (int32_t)sizeof(Tracker<float>::RefitOut); }
void oracle_get_refits(void *hv, void *dst) {
    Handle *h = (Handle *)hv;
    if (h->useDouble) copy_out(dst, h->d->refits.data(), h->d->refits.size() * sizeof(Tracker<double>::RefitOut));
    else copy_out(dst, h->f->refits.data(), h->f->refits.size() * sizeof(Tracker<float>::RefitOut));
}
/* primitives for the pins: rotate a state (x[1], p[5], c[15]) by beta; chi2 of d with covariance S (15) */
int oracle_rotate(int use_double, double *x, double *p, double *c, double beta, double CB, double smax) {
    auto run = [&](auto tag) {
        using T = decltype(tag);
        State<T> st; st.x = T(*x); st.chi2 = T(0); st.nfit = 0;
        for (int i = 0; i < 5; i++) st.p[i] = T(p[i]);
        for (int i = 0, k = 0; i < 5; i++) for (int j = 0; j <= i; j++) { st.C[i][j] = st.C[j][i] = T(c[k++]); }
        if (!rotate(st, T(std::cos(beta)), T(std::sin(beta)), T(CB), T(smax))) return 0;
        *x = double(st.x);
        for (int i = 0; i < 5; i++) p[i] = double(st.p[i]);
        for (int i = 0, k = 0; i < 5; i++) for (int j = 0; j <= i; j++) c[k++] = double(st.C[i][j]);
        return 1;
    };
    return use_double ? run(double(0)) : run(float(0));
}
double oracle_chi2_5(int use_double, const double *d, const double *s15) {
    auto run = [&](auto tag) {
        using T = decltype(tag);
        T dd[5], S[5][5];
        for (int i = 0; i < 5; i++) dd[i] = T(d[i]);
        for (int i = 0, k = 0; i < 5; i++) for (int j = 0; j <= i; j++) { S[i][j] = S[j][i] = T(s15[k++]); }
        return double(chi2_5(dd, S));
    };
    return use_double ? run(double(0)) : run(float(0));
}

int oracle_propagate(int use_double, double *x, double *p, double *c, double x2, double CB, double smax, double *J) {
    return use_double ? propagate_c<double>(x, p, c, x2, CB, smax, J) : propagate_c<float>(x, p, c, x2, CB, smax, J);
}
void oracle_update(int use_double, double *p, double *c, double *chi2, int coord, double m, double e2) {
    if (use_double) update_c<double>(p, c, chi2, coord, m, e2); else update_c<float>(p, c, chi2, coord, m, e2);
}

}  /* extern "C" */
