// Host-side tables: quadrature, harmonics, schedules.  See host_tables.h.
#include "host_tables.h"

#include <algorithm>
#include <array>
#include <cmath>

namespace doctors {

namespace {

typedef long double real;

struct LqSystem {
    int n = 0;                               // levels per axis = N/2
    std::vector<std::array<int, 3>> pts;     // 1-based level triples of one octant
    std::vector<std::array<int, 3>> classes; // sorted triples = weight classes
    std::vector<int> cls_of;                 // class index per point
};

LqSystem lq_structure(int N)
{
    LqSystem s;
    s.n = N / 2;
    for (int i = 1; i <= s.n; ++i)
        for (int j = 1; j <= s.n; ++j) {
            int k = s.n + 2 - i - j;
            if (k >= 1 && k <= s.n) s.pts.push_back({i, j, k});
        }
    for (auto p : s.pts) {
        std::sort(p.begin(), p.end());
        if (std::find(s.classes.begin(), s.classes.end(), p) == s.classes.end()) s.classes.push_back(p);
    }
    std::sort(s.classes.begin(), s.classes.end());
    for (auto p : s.pts) {
        std::sort(p.begin(), p.end());
        s.cls_of.push_back(int(std::find(s.classes.begin(), s.classes.end(), p) - s.classes.begin()));
    }
    return s;
}

// Dense solve with partial pivoting; returns false if singular.
bool solve_dense(std::vector<std::vector<real>>& A, std::vector<real>& b)
{
    int m = int(b.size());
    for (int c = 0; c < m; ++c) {
        int piv = c;
        for (int r = c + 1; r < m; ++r)
            if (fabsl(A[r][c]) > fabsl(A[piv][c])) piv = r;
        if (fabsl(A[piv][c]) < 1e-30L) return false;
        std::swap(A[piv], A[c]);
        std::swap(b[piv], b[c]);
        for (int r = c + 1; r < m; ++r) {
            real f = A[r][c] / A[c][c];
            for (int cc = c; cc < m; ++cc) A[r][cc] -= f * A[c][cc];
            b[r] -= f * b[c];
        }
    }
    for (int r = m - 1; r >= 0; --r) {
        real s = b[r];
        for (int cc = r + 1; cc < m; ++cc) s -= A[r][cc] * b[cc];
        b[r] = s / A[r][r];
    }
    return true;
}

// For a trial mu_1^2: levels, class weights (octant-normalised) from the even one-axis moment
// conditions sum w mu_x^{2k} = 1/(2k+1), k = 0, 2, 3, .., n-1 (k = 1 follows from k = 0 by
// symmetry), plus for N = 16 the mixed condition sum w (mu eta xi)^4 = 1/5005.  Returns the
// residual of the k = n condition, which fixes mu_1.
bool lq_weights(const LqSystem& s, int N, real mu1sq, std::vector<real>& mu, std::vector<real>& wc, real& resid)
{
    int n = s.n, nc = int(s.classes.size());
    mu.assign(n, 0);
    real step = N > 2 ? 2.0L * (1.0L - 3.0L * mu1sq) / (N - 2) : 0.0L;
    for (int i = 0; i < n; ++i) mu[i] = sqrtl(mu1sq + i * step);
    std::vector<int> ks;
    ks.push_back(0);
    for (int k = 2; k <= n - 1; ++k) ks.push_back(k);
    int neq = int(ks.size()) + (N == 16 ? 1 : 0);
    if (neq != nc) return false;
    std::vector<std::vector<real>> A(nc, std::vector<real>(nc, 0));
    std::vector<real> b(nc, 0);
    for (size_t e = 0; e < ks.size(); ++e) {
        for (size_t p = 0; p < s.pts.size(); ++p) A[e][s.cls_of[p]] += powl(mu[s.pts[p][0] - 1], 2 * ks[e]);
        b[e] = 1.0L / (2 * ks[e] + 1);
    }
    if (N == 16) {
        for (size_t p = 0; p < s.pts.size(); ++p) {
            real t = mu[s.pts[p][0] - 1] * mu[s.pts[p][1] - 1] * mu[s.pts[p][2] - 1];
            A[nc - 1][s.cls_of[p]] += t * t * t * t;
        }
        b[nc - 1] = 1.0L / 5005.0L;
    }
    if (!solve_dense(A, b)) return false;
    wc = b;
    real r = 0;
    for (size_t p = 0; p < s.pts.size(); ++p) r += wc[s.cls_of[p]] * powl(mu[s.pts[p][0] - 1], 2 * n);
    resid = r - 1.0L / (2 * n + 1);
    return true;
}

}  // namespace

bool level_symmetric(int N, std::vector<double>& omega, std::vector<double>& w)
{
    if (!(N == 2 || N == 4 || N == 6 || N == 8 || N == 12 || N == 16)) return false;
    LqSystem s = lq_structure(N);
    std::vector<real> mu, wc;
    real resid = 0;
    if (N == 2) {
        mu.assign(1, sqrtl(1.0L / 3.0L));
        wc.assign(1, 1.0L);
    } else {
        // scan (0, 1/3) for sign changes of the k = n residual, bisect each, keep the root whose
        // weights are all positive (S6 has a second root with a negative weight)
        const int NS = 4000;
        real lo = 1e-3L, hi = 1.0L / 3.0L - 1e-4L;
        bool have = false;
        real best = 0;
        real xprev = lo, fprev = 0;
        bool okprev = lq_weights(s, N, xprev, mu, wc, fprev);
        for (int t = 1; t <= NS; ++t) {
            real x = lo + (hi - lo) * t / NS, f = 0;
            bool ok = lq_weights(s, N, x, mu, wc, f);
            if (ok && okprev && ((fprev < 0) != (f < 0))) {
                real a = xprev, fa = fprev, c = x;
                for (int it = 0; it < 200; ++it) {
                    real m = 0.5L * (a + c), fm = 0;
                    if (!lq_weights(s, N, m, mu, wc, fm)) break;
                    if ((fm < 0) == (fa < 0)) { a = m; fa = fm; } else { c = m; }
                }
                real root = 0.5L * (a + c), fr = 0;
                if (lq_weights(s, N, root, mu, wc, fr) && fabsl(fr) < 1e-13L &&
                    *std::min_element(wc.begin(), wc.end()) > 0) {
                    have = true;
                    best = root;
                }
            }
            xprev = x; fprev = f; okprev = ok;
        }
        if (!have) return false;
        lq_weights(s, N, best, mu, wc, resid);
    }
    int M = int(s.pts.size());
    omega.assign(size_t(8) * M * 3, 0.0);
    w.assign(size_t(8) * M, 0.0);
    const real pi = acosl(-1.0L);
    for (int o = 0; o < 8; ++o)
        for (int p = 0; p < M; ++p) {
            size_t n = size_t(o) * M + p;
            omega[3 * n + 0] = double((o & 1 ? -1 : 1) * mu[s.pts[p][0] - 1]);
            omega[3 * n + 1] = double((o & 2 ? -1 : 1) * mu[s.pts[p][1] - 1]);
            omega[3 * n + 2] = double((o & 4 ? -1 : 1) * mu[s.pts[p][2] - 1]);
            w[n] = double(wc[s.cls_of[p]] * 4.0L * pi / 8.0L);
        }
    return true;
}

void real_harmonics(int L, double mu, double eta, double xi, double* Y)
{
    // Cartesian forms of the R4 convention (lm = l^2 + l + m)
    Y[0] = 1.0;
    if (L < 1) return;
    Y[1] = eta; Y[2] = xi; Y[3] = mu;
    if (L < 2) return;
    const double s3 = std::sqrt(3.0);
    Y[4] = s3 * mu * eta;
    Y[5] = s3 * xi * eta;
    Y[6] = 0.5 * (3.0 * xi * xi - 1.0);
    Y[7] = s3 * xi * mu;
    Y[8] = 0.5 * s3 * (mu * mu - eta * eta);
    if (L < 3) return;
    const double a = std::sqrt(5.0 / 8.0), b = std::sqrt(15.0), c = std::sqrt(3.0 / 8.0);
    Y[9]  = a * (3.0 * mu * mu * eta - eta * eta * eta);
    Y[10] = b * xi * mu * eta;
    Y[11] = c * (5.0 * xi * xi - 1.0) * eta;
    Y[12] = 0.5 * (5.0 * xi * xi * xi - 3.0 * xi);
    Y[13] = c * (5.0 * xi * xi - 1.0) * mu;
    Y[14] = 0.5 * b * xi * (mu * mu - eta * eta);
    Y[15] = a * (mu * mu * mu - 3.0 * mu * eta * eta);
}

void projection_tables(int L, const std::vector<double>& omega, const std::vector<double>& w,
                       std::vector<double>& Mtab, std::vector<double>& Dtab)
{
    int nm = (L + 1) * (L + 1);
    size_t nd = w.size();
    Mtab.assign(nd * nm, 0.0);
    Dtab.assign(nd * nm, 0.0);
    const double pi = std::acos(-1.0);
    double Y[16];
    for (size_t n = 0; n < nd; ++n) {
        real_harmonics(L, omega[3 * n], omega[3 * n + 1], omega[3 * n + 2], Y);
        for (int l = 0; l <= L; ++l)
            for (int m = -l; m <= l; ++m) {
                int lm = l * l + l + m;
                Mtab[n * nm + lm] = (2 * l + 1) / (4.0 * pi) * Y[lm];
                Dtab[n * nm + lm] = w[n] * Y[lm];
            }
    }
}

long long wavefront_size(int nx, int ny, int nz, int S)
{
    // Eq. (9): C(S) minus the three single-axis overflows plus the three pair overlaps.
    auto T = [](long long d) { return d > 0 ? d * (d + 1) / 2 : 0LL; };   // triangular number of max(d,0)
    long long s1 = (long long)S + 1;
    return T(s1) - T(s1 - nx) - T(s1 - ny) - T(s1 - nz) + T(s1 - nx - ny) + T(s1 - ny - nz) + T(s1 - nx - nz);
}

void subsweep_schedule(int nx, int ny, int nz, int octant,
                       std::vector<int32_t>& plane_offset, std::vector<int32_t>& cell_of)
{
    int planes = nx + ny + nz - 2;
    plane_offset.assign(planes + 1, 0);
    cell_of.assign(size_t(nx) * ny * nz, 0);
    size_t cnt = 0;
    for (int S = 0; S < planes; ++S) {
        plane_offset[S] = int32_t(cnt);
        // Eq. (8): i'+j'+k' = S inside the box; Table 1 order: i' descending, then j' descending
        int ihi = std::min(S, nx - 1), ilo = std::max(0, S - (ny - 1) - (nz - 1));
        for (int ip = ihi; ip >= ilo; --ip) {
            int r = S - ip;
            int jhi = std::min(r, ny - 1), jlo = std::max(0, r - (nz - 1));
            for (int jp = jhi; jp >= jlo; --jp) {
                int kp = r - jp;
                int i = (octant & 1) ? nx - 1 - ip : ip;
                int j = (octant & 2) ? ny - 1 - jp : jp;
                int k = (octant & 4) ? nz - 1 - kp : kp;
                cell_of[cnt++] = int32_t(i + nx * (j + ny * k));
            }
        }
    }
    plane_offset[planes] = int32_t(cnt);
}

}  // namespace doctors
