/* ORACLE — test infrastructure, not product code.
 *
 * Plain fp64 CPU implementation of the DOCTORS hot path, written from the paper
 * and the readings in DESIGN.md / SURVEY.md §8(c).  It shares no
 * code with the CUDA library.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * What is here (each function cites the passage it follows):
 *   orc_wavefront_size   P(S), Eqs. (9)-(22)
 *   orc_schedule         sub-sweep membership and order, PAPER.md:72-81 (Eq. 8), Table 1 (:121-139)
 *   orc_sweep            one transport sweep of Eq. (2) over all directions,
 *                        diamond difference, vacuum boundaries (:37),
 *                        scalar flux / moments by Eq. (3) (:39)
 *   orc_raytrace         uncollided fluence of Eq. (4) by exact voxel ray tracing
 *
 * Layouts: cell c = i + nx*(j + ny*k) (x fastest); moments [nm][cells]; all double.
 * Threads (OpenMP) split independent directions / rays only; every sum that
 * crosses threads is done in a fixed order, so results do not depend on the
 * thread count.
 */
#define _USE_MATH_DEFINES
#define _GNU_SOURCE
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---- PAPER.md:85-117, Eqs. (9)-(22): number of voxels in sub-sweep S ---- */
static int64_t tri(int64_t d) { return d * (d + 1) / 2; }
static int64_t pos(int64_t v) { return v > 0 ? v : 0; }

int64_t orc_wavefront_size(int nx, int ny, int nz, int S)
{
    int64_t Cs  = (int64_t)(S + 1) * (S + 2) / 2;              /* Eq. (10) */
    int64_t dx  = pos((int64_t)S + 1 - nx);                    /* Eq. (17) */
    int64_t dy  = pos((int64_t)S + 1 - ny);                    /* Eq. (18), "d_v" read as d_y */
    int64_t dz  = pos((int64_t)S + 1 - nz);                    /* Eq. (19) */
    int64_t dxy = pos((int64_t)S + 1 - nx - ny);               /* Eq. (20) */
    int64_t dyz = pos((int64_t)S + 1 - ny - nz);               /* Eq. (21) */
    int64_t dxz = pos((int64_t)S + 1 - nx - nz);               /* Eq. (22) */
    return Cs - tri(dx) - tri(dy) - tri(dz) + tri(dxy) + tri(dyz) + tri(dxz);   /* Eq. (9), (11)-(16) */
}

/* ---- PAPER.md:72-81 Eq. (8) + Table 1: cells of every sub-sweep, in Table 1 order ----
 * Sweep-space indices (i',j',k') with i'+j'+k' = S, 0 <= i' < nx etc.  Table 1 lists
 * i' descending, then j' descending.  Octant bit0/1/2 set = sweep runs in -x/-y/-z,
 * so the mesh index is mirrored: i = nx-1-i'.
 * plane_offset has nx+ny+nz-1 entries, cell_of has nx*ny*nz. */
void orc_schedule(int nx, int ny, int nz, int octant, int32_t *plane_offset, int32_t *cell_of)
{
    int planes = nx + ny + nz - 2;
    int64_t n = 0;
    for (int S = 0; S < planes; ++S) {
        plane_offset[S] = (int32_t)n;
        for (int ip = (S < nx - 1 ? S : nx - 1); ip >= 0; --ip) {
            for (int jp = (S - ip < ny - 1 ? S - ip : ny - 1); jp >= 0; --jp) {
                int kp = S - ip - jp;
                if (kp >= nz) break;                 /* smaller j' only makes k' larger */
                int i = (octant & 1) ? nx - 1 - ip : ip;
                int j = (octant & 2) ? ny - 1 - jp : jp;
                int k = (octant & 4) ? nz - 1 - kp : kp;
                cell_of[n++] = (int32_t)(i + nx * (j + ny * k));
            }
        }
    }
    plane_offset[planes] = (int32_t)n;
}

/* ---- one cell, one direction: diamond difference (textbook DD of ref. 13) ----
 * Balance over the cell + psi_c = (psi_in + psi_out)/2 on each axis:
 *   psi_c = (q + cx*pin_x + cy*pin_y + cz*pin_z) / (sigt + cx + cy + cz),  c_d = 2|Omega_d|/Delta_d
 *   pout_d = 2 psi_c - pin_d
 * closure 1 (reading R2): any outflow < 0 is set to 0 and the balance is re-solved with that
 * face's DD relation dropped; repeat while new faces flip (at most 3 rounds). */
static inline double dd_cell(double q, double sigt, const double c[3], const double pin[3],
                             int closure, double pout[3], int64_t *nfix)
{
    int fixed[3] = {0, 0, 0};
    double psi = 0.0;
    for (int pass = 0; pass < 4; ++pass) {
        double num = q, den = sigt;
        for (int d = 0; d < 3; ++d) {
            if (fixed[d]) num += 0.5 * c[d] * pin[d];
            else { num += c[d] * pin[d]; den += c[d]; }
        }
        psi = num / den;
        int flipped = 0;
        for (int d = 0; d < 3; ++d) {
            pout[d] = fixed[d] ? 0.0 : 2.0 * psi - pin[d];
            if (closure == 1 && !fixed[d] && pout[d] < 0.0) { fixed[d] = 1; flipped = 1; }
        }
        if (!flipped) break;
        if (nfix) ++*nfix;
    }
    for (int d = 0; d < 3; ++d) if (fixed[d]) pout[d] = 0.0;
    return psi;
}

/* sweep one direction in lexicographic upwind order; psi[cells] out; returns leakage
 * sum over outflow boundary faces of |Omega_d| * A_d * psi_out  (not yet weighted by w_n). */
static double sweep_dir_lex(int nx, int ny, int nz, const double del[3], const double *sigt,
                            const double *qn, const double om[3], int closure,
                            double *psi, int64_t *nfix)
{
    double c[3] = {2.0 * fabs(om[0]) / del[0], 2.0 * fabs(om[1]) / del[1], 2.0 * fabs(om[2]) / del[2]};
    double area[3] = {del[1] * del[2], del[0] * del[2], del[0] * del[1]};
    double *fy = (double *)calloc((size_t)nx, sizeof(double));
    double *fz = (double *)calloc((size_t)nx * ny, sizeof(double));
    double leak = 0.0;
    for (int kp = 0; kp < nz; ++kp) {
        int k = om[2] > 0 ? kp : nz - 1 - kp;
        for (int ip = 0; ip < nx; ++ip) fy[ip] = 0.0;           /* vacuum inflow on the y face (:37) */
        for (int jp = 0; jp < ny; ++jp) {
            int j = om[1] > 0 ? jp : ny - 1 - jp;
            double fx = 0.0;                                      /* vacuum inflow on the x face */
            for (int ip = 0; ip < nx; ++ip) {
                int i = om[0] > 0 ? ip : nx - 1 - ip;
                size_t cidx = (size_t)i + (size_t)nx * (j + (size_t)ny * k);
                double pin[3] = {fx, fy[i], kp == 0 ? 0.0 : fz[i + (size_t)nx * j]};
                double pout[3];
                psi[cidx] = dd_cell(qn[cidx], sigt[cidx], c, pin, closure, pout, nfix);
                fx = pout[0]; fy[i] = pout[1]; fz[i + (size_t)nx * j] = pout[2];
                if (ip == nx - 1) leak += fabs(om[0]) * area[0] * pout[0];
                if (jp == ny - 1) leak += fabs(om[1]) * area[1] * pout[1];
                if (kp == nz - 1) leak += fabs(om[2]) * area[2] * pout[2];
            }
        }
    }
    free(fy); free(fz);
    return leak;
}

/* same direction, but cells visited in the paper's sub-sweep order (Eq. 8 / Table 1).
 * Each cell reads its three upwind neighbours' outflows from full per-cell face arrays. */
static double sweep_dir_hyperplane(int nx, int ny, int nz, const double del[3], const double *sigt,
                                   const double *qn, const double om[3], int closure,
                                   double *psi, int64_t *nfix)
{
    size_t cells = (size_t)nx * ny * nz;
    int octant = (om[0] < 0 ? 1 : 0) | (om[1] < 0 ? 2 : 0) | (om[2] < 0 ? 4 : 0);
    int planes = nx + ny + nz - 2;
    int32_t *off = (int32_t *)malloc(sizeof(int32_t) * (planes + 1));
    int32_t *cell_of = (int32_t *)malloc(sizeof(int32_t) * cells);
    double *ox = (double *)malloc(sizeof(double) * cells * 3), *oy = ox + cells, *oz = oy + cells;
    orc_schedule(nx, ny, nz, octant, off, cell_of);
    double c[3] = {2.0 * fabs(om[0]) / del[0], 2.0 * fabs(om[1]) / del[1], 2.0 * fabs(om[2]) / del[2]};
    double area[3] = {del[1] * del[2], del[0] * del[2], del[0] * del[1]};
    int sx = om[0] > 0 ? 1 : -1, sy = om[1] > 0 ? 1 : -1, sz = om[2] > 0 ? 1 : -1;
    double leak = 0.0;
    for (int S = 0; S < planes; ++S)
        for (int32_t t = off[S]; t < off[S + 1]; ++t) {
            size_t cidx = (size_t)cell_of[t];
            int i = (int)(cidx % nx), j = (int)((cidx / nx) % ny), k = (int)(cidx / ((size_t)nx * ny));
            int iu = i - sx, ju = j - sy, ku = k - sz;               /* upwind neighbours */
            double pin[3];
            pin[0] = (iu < 0 || iu >= nx) ? 0.0 : ox[(size_t)iu + (size_t)nx * (j + (size_t)ny * k)];
            pin[1] = (ju < 0 || ju >= ny) ? 0.0 : oy[(size_t)i + (size_t)nx * (ju + (size_t)ny * k)];
            pin[2] = (ku < 0 || ku >= nz) ? 0.0 : oz[(size_t)i + (size_t)nx * (j + (size_t)ny * ku)];
            double pout[3];
            psi[cidx] = dd_cell(qn[cidx], sigt[cidx], c, pin, closure, pout, nfix);
            ox[cidx] = pout[0]; oy[cidx] = pout[1]; oz[cidx] = pout[2];
            if (i + sx < 0 || i + sx >= nx) leak += fabs(om[0]) * area[0] * pout[0];
            if (j + sy < 0 || j + sy >= ny) leak += fabs(om[1]) * area[1] * pout[1];
            if (k + sz < 0 || k + sz >= nz) leak += fabs(om[2]) * area[2] * pout[2];
        }
    free(off); free(cell_of); free(ox);
    return leak;
}

/* ---- one sweep of Eq. (2) over all directions; moments by Eq. (3) ----
 * Q    [nm][cells]  source moments (4pi-integrated convention, reading R6)
 * Mtab [ndir][nm]   (2l+1)/(4pi) Y_lm(Omega_n)       -> q_n = sum_lm Mtab[n][lm] Q_lm   (Eq. 2 rhs, moment form R3)
 * Dtab [nm][ndir]   w_n Y_lm(Omega_n)                -> phi_lm += Dtab[lm][n] psi_n     (Eq. 3)
 * Directions are ordered octant-major (octant o = n / (ndir/8)).  Every direction is independent of the others
 * (PAPER.md:119 discusses exactly this), so they are computed in batches of whole octants, one thread per
 * direction; phi_lm(c) is then summed over the directions of the batch in index order, batches in order: for
 * every (lm, c) the terms are added in the order n = 0, 1, ..., ndir-1 whatever the batch size and the
 * thread count are (the batch only bounds the memory held for psi_n: 6 GiB).
 * order: 0 lexicographic loops, 1 the paper's sub-sweep order.
 * psi_all: NULL or [ndir][cells] (angular flux, for tests).
 * leak_out: sum_n w_n * leakage_n.   nfix_out: NULL or fix-up event count. */
void orc_sweep(int nx, int ny, int nz, double dx, double dy, double dz,
               const double *sigt, const double *Q, int nm,
               int ndir, const double *omega, const double *w,
               const double *Mtab, const double *Dtab,
               int closure, int order,
               double *phi, double *leak_out, double *psi_all, int64_t *nfix_out, int nthreads)
{
    size_t cells = (size_t)nx * ny * nz;
    double del[3] = {dx, dy, dz};
    int per_oct = ndir / 8 > 0 && ndir % 8 == 0 ? ndir / 8 : ndir;
    int chunk = per_oct;                                            /* directions per batch: whole octants */
    while (chunk + per_oct <= ndir && (double)cells * (chunk + per_oct) * 16.0 <= 6.0 * 1073741824.0) chunk += per_oct;
    double *psi_buf = (double *)malloc(sizeof(double) * cells * chunk);
    double *qn_buf = (double *)malloc(sizeof(double) * cells * chunk);
    double *leak_n = (double *)calloc((size_t)ndir, sizeof(double));
    int64_t *nfix_n = (int64_t *)calloc((size_t)ndir, sizeof(int64_t));
    memset(phi, 0, sizeof(double) * cells * nm);
    if (nthreads < 1) nthreads = 1;
    const int64_t cblock = 2048;                                    /* cells handled by one thread at a time in the moment sums */
    int64_t nblocks = ((int64_t)cells + cblock - 1) / cblock;
    for (int n0 = 0; n0 < ndir; n0 += chunk) {
        int nb = n0 + chunk <= ndir ? chunk : ndir - n0;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
        for (int m = 0; m < nb; ++m) {
            int n = n0 + m;
            double *qn = qn_buf + cells * m, *psi = psi_buf + cells * m;
            for (size_t c = 0; c < cells; ++c) {
                double q = 0.0;
                for (int lm = 0; lm < nm; ++lm) q += Mtab[(size_t)n * nm + lm] * Q[(size_t)lm * cells + c];
                qn[c] = q;
            }
            if (order == 0) leak_n[n] = sweep_dir_lex(nx, ny, nz, del, sigt, qn, omega + 3 * n, closure, psi, nfix_n + n);
            else leak_n[n] = sweep_dir_hyperplane(nx, ny, nz, del, sigt, qn, omega + 3 * n, closure, psi, nfix_n + n);
            if (psi_all) memcpy(psi_all + cells * n, psi, sizeof(double) * cells);
        }
#pragma omp parallel for schedule(static) num_threads(nthreads)
        for (int64_t blk = 0; blk < nblocks; ++blk) {                /* independent cells: any split gives the same sums */
            size_t c0 = (size_t)(blk * cblock), c1 = c0 + (size_t)cblock < cells ? c0 + (size_t)cblock : cells;
            for (int lm = 0; lm < nm; ++lm)
                for (int m = 0; m < nb; ++m) {                      /* Eq. (3): fixed direction order */
                    double d = Dtab[(size_t)lm * ndir + n0 + m];
                    const double *psi = psi_buf + cells * m;
                    double *p = phi + (size_t)lm * cells;
                    for (size_t c = c0; c < c1; ++c) p[c] += d * psi[c];
                }
        }
    }
    double leak = 0.0;
    int64_t nf = 0;
    for (int n = 0; n < ndir; ++n) { leak += w[n] * leak_n[n]; nf += nfix_n[n]; }
    if (leak_out) *leak_out = leak;
    if (nfix_out) *nfix_out = nf;
    free(psi_buf); free(qn_buf); free(leak_n); free(nfix_n);
}

static int cmp_double(const void *a, const void *b)
{
    double x = *(const double *)a, y = *(const double *)b;
    return (x > y) - (x < y);
}

/* ---- PAPER.md:44-49 Eq. (4): uncollided fluence by ray tracing (reading R11, R12) ----
 * For every cell centre r_c:  d = r_c - r_s, R = |d|, u = d/R.
 *   kind 2 (cone): u . axis >= cos_half, else phi_u = 0.
 *   kind 3 (fan, "two additional parameters, phi and theta, describe the azimuthal and polar
 *   angles subtended by the fan"; reading R18): with a = axis / |axis|, n = fan_n (unit normal of the fan plane,
 *   perpendicular to a) and t = n x a, the direction u has the polar angle beta = asin(u . n) out of the plane
 *   and the azimuth alpha = atan2(u . t, u . a) in it; lit iff |beta| <= half2 and |alpha| <= half, i.e.
 *   |u . n| <= sin_half2 and u . a >= cos_half * sqrt((u . a)^2 + (u . t)^2).  Hard edges, 4 pi kept (R12).
 *   The segment [0,R] is clipped to the mesh box (outside is vacuum), cut at every grid plane it crosses (crossing
 *   parameters computed plane by plane, then sorted) and every piece is assigned to the voxel its midpoint lies in.  The
 *   library's kernel walks the same path incrementally (running tMax / tDelta per axis): the two agree to rounding, and
 *   an error in either traversal shows up in the comparison.  Per material m the areal density A_m = sum rho * length
 *   is accumulated (independent of the group), then
 *     tau_g = sum_m sigt_hat[m][g] A_m,   phi_u^g = S_g exp(-tau_g) / (4 pi R^2).
 * mesh centred on the origin.  phi_u [G][cells]; areal NULL or [n_mat][cells]. */
void orc_raytrace(int nx, int ny, int nz, double dx, double dy, double dz,
                  const uint8_t *mat, const double *rho, int n_mat, int G, const double *sigt_hat,
                  int kind, const double *spos, const double *axis, double cos_half,
                  const double *spectrum, double *phi_u, double *areal, int nthreads,
                  const double *fan_n, double sin_half2)
{
    size_t cells = (size_t)nx * ny * nz;
    int nn[3] = {nx, ny, nz};
    double del[3] = {dx, dy, dz};
    double lo[3] = {-0.5 * nx * dx, -0.5 * ny * dy, -0.5 * nz * dz};
    double an = sqrt(axis[0] * axis[0] + axis[1] * axis[1] + axis[2] * axis[2]);
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for schedule(static) num_threads(nthreads)
    for (int64_t cc = 0; cc < (int64_t)cells; ++cc) {
        size_t c = (size_t)cc;
        int ci[3] = {(int)(c % nx), (int)((c / nx) % ny), (int)(c / ((size_t)nx * ny))};
        double rc[3], d[3], u[3], R2 = 0.0;
        double A[16];
        for (int m = 0; m < n_mat; ++m) A[m] = 0.0;
        for (int a = 0; a < 3; ++a) { rc[a] = lo[a] + (ci[a] + 0.5) * del[a]; d[a] = rc[a] - spos[a]; R2 += d[a] * d[a]; }
        double R = sqrt(R2);
        for (int a = 0; a < 3; ++a) u[a] = d[a] / R;
        int lit = 1;
        if (kind == 2) {
            double ca = (u[0] * axis[0] + u[1] * axis[1] + u[2] * axis[2]) / an;
            if (ca < cos_half) lit = 0;
        }
        if (kind == 3) {
            double a[3] = {axis[0] / an, axis[1] / an, axis[2] / an};
            double t[3] = {fan_n[1] * a[2] - fan_n[2] * a[1], fan_n[2] * a[0] - fan_n[0] * a[2], fan_n[0] * a[1] - fan_n[1] * a[0]};
            double ua = u[0] * a[0] + u[1] * a[1] + u[2] * a[2];
            double un = u[0] * fan_n[0] + u[1] * fan_n[1] + u[2] * fan_n[2];
            double ut = u[0] * t[0] + u[1] * t[1] + u[2] * t[2];
            if (fabs(un) > sin_half2) lit = 0;
            if (ua < cos_half * sqrt(ua * ua + ut * ut)) lit = 0;
        }
        if (lit) {
            /* The radiological path written out as its definition (reading R11): the part of the segment [0, R] inside the
             * mesh box is cut at EVERY grid plane it crosses, x, y and z planes alike; the crossing parameters are computed
             * one by one from the plane positions and sorted; each piece between two consecutive crossings lies in one voxel,
             * found from the piece's midpoint, and adds rho * length to that voxel's material.  (No incremental stepping,
             * no running tMax / tDelta, no tie-breaking: a ray through a voxel edge gives a zero-length piece.) */
            double t0 = 0.0, t1 = R;                                /* in-box interval by slab clipping */
            for (int a = 0; a < 3; ++a) {
                double hi_a = lo[a] + nn[a] * del[a];
                if (u[a] != 0.0) {
                    double ta = (lo[a] - spos[a]) / u[a], tb = (hi_a - spos[a]) / u[a];
                    double tnear = ta < tb ? ta : tb, tfar = ta < tb ? tb : ta;
                    if (tnear > t0) t0 = tnear;
                    if (tfar < t1) t1 = tfar;
                } else if (spos[a] < lo[a] || spos[a] > hi_a) t1 = -1.0;   /* parallel to the slab and outside it */
            }
            if (t1 > t0) {
                double *tc = (double *)malloc(sizeof(double) * (size_t)(nx + ny + nz + 8));
                int n = 0;
                tc[n++] = t0;
                for (int a = 0; a < 3; ++a) {
                    if (u[a] == 0.0) continue;
                    /* planes between the two end points of the in-box piece (one spare on each side) */
                    double pa = (spos[a] + t0 * u[a] - lo[a]) / del[a], pb = (spos[a] + t1 * u[a] - lo[a]) / del[a];
                    int p_lo = (int)floor(pa < pb ? pa : pb) - 1, p_hi = (int)ceil(pa < pb ? pb : pa) + 1;
                    if (p_lo < 0) p_lo = 0;
                    if (p_hi > nn[a]) p_hi = nn[a];
                    for (int pl = p_lo; pl <= p_hi; ++pl) {
                        double t = (lo[a] + pl * del[a] - spos[a]) / u[a];
                        if (t > t0 && t < t1) tc[n++] = t;
                    }
                }
                tc[n++] = t1;
                qsort(tc, (size_t)n, sizeof(double), cmp_double);
                for (int i = 0; i + 1 < n; ++i) {
                    double len = tc[i + 1] - tc[i];
                    if (!(len > 0.0)) continue;
                    double tm = 0.5 * (tc[i] + tc[i + 1]);
                    int vi[3];
                    for (int a = 0; a < 3; ++a) {
                        int ii = (int)floor((spos[a] + tm * u[a] - lo[a]) / del[a]);
                        if (ii < 0) ii = 0;
                        if (ii > nn[a] - 1) ii = nn[a] - 1;
                        vi[a] = ii;
                    }
                    size_t v = (size_t)vi[0] + (size_t)nx * (vi[1] + (size_t)ny * vi[2]);
                    A[mat[v]] += rho[v] * len;
                }
                free(tc);
            }
        }
        for (int m = 0; m < n_mat && areal; ++m) areal[(size_t)m * cells + c] = A[m];
        for (int g = 0; g < G; ++g) {
            double tau = 0.0;
            for (int m = 0; m < n_mat; ++m) tau += sigt_hat[(size_t)m * G + g] * A[m];
            phi_u[(size_t)g * cells + c] = lit ? spectrum[g] * exp(-tau) / (4.0 * M_PI * R2) : 0.0;
        }
    }
}
