// Streaming kernels of the hot path: ray trace (a1), fixed source (a2), iteration update and
// convergence check (a6), and the paper's own one-launch-per-sub-sweep sweep (sweep_mode 1).
#pragma once
#include "device_common.cuh"

namespace doctors {

// =========================================================================================
// a1  Uncollided fluence, Eq. (4) (PAPER.md:44-49; "ray-tracing", :68 "straightforward").
// One thread per (cell, source).  The segment source -> cell centre is clipped to the mesh
// box (outside is vacuum) and walked voxel by voxel with a parametric traversal; the areal
// density rho*length is accumulated PER MATERIAL (group independent), then for every group
//   tau_g = sum_m sigt_hat[m][g] A_m,   phi_u^g = S_g exp(-tau_g) / (4 pi R^2)   (reading R12).
// Geometry and the exponent are fp64 (cheap here, keeps tie-breaks stable); output is fp32.
// =========================================================================================
constexpr int kRayThreads = 128;

__global__ void __launch_bounds__(kRayThreads)
k_raytrace(MeshDev m, const uint8_t* __restrict__ mat /*dense [nz][ny][nx]*/, const float* __restrict__ rho /*dense*/,
           const SourceDev* __restrict__ srcs, int src0, const double* __restrict__ sigt_hat,
           const double* __restrict__ spectrum, int n_mat, int G, float* __restrict__ phi_u)
{
    __shared__ double sA[kMaxMaterials][kRayThreads];
    const int s = blockIdx.y;
    const SourceDev src = srcs[src0 + s];
    long long cp = (long long)blockIdx.x * kRayThreads + threadIdx.x;
    if (cp >= m.cells_p) return;
    int i, j, k;
    const bool real = cell_ijk(m, cp, i, j, k);
    float* out = phi_u + (size_t)s * G * m.cells_p + cp;
    if (!real || src.kind == 0) {
        for (int g = 0; g < G; ++g) out[(size_t)g * m.cells_p] = 0.0f;
        return;
    }
    const int tid = threadIdx.x;
    for (int q = 0; q < n_mat; ++q) sA[q][tid] = 0.0;
    const int nn[3] = {m.nx, m.ny, m.nz};
    const double del[3] = {m.dx, m.dy, m.dz};
    const double lo[3] = {m.x0 - 0.5 * m.dx, m.y0 - 0.5 * m.dy, m.z0 - 0.5 * m.dz};
    const double rc[3] = {m.x0 + i * m.dx, m.y0 + j * m.dy, m.z0 + k * m.dz};
    double d[3], u[3], R2 = 0.0;
#pragma unroll
    for (int a = 0; a < 3; ++a) { d[a] = rc[a] - src.pos[a]; R2 += d[a] * d[a]; }
    const double R = sqrt(R2);
#pragma unroll
    for (int a = 0; a < 3; ++a) u[a] = d[a] / R;
    bool lit = true;
    if (src.kind == 2) lit = (u[0] * src.axis[0] + u[1] * src.axis[1] + u[2] * src.axis[2]) >= src.cos_half;
    if (src.kind == 3) {
        // fan beam (reading R18): polar angle out of the fan plane |beta| <= half2, azimuth in the plane |alpha| <= half
        const double* a = src.axis; const double* nv = src.fan_n;
        const double tv[3] = {nv[1] * a[2] - nv[2] * a[1], nv[2] * a[0] - nv[0] * a[2], nv[0] * a[1] - nv[1] * a[0]};
        const double ua = u[0] * a[0] + u[1] * a[1] + u[2] * a[2], un = u[0] * nv[0] + u[1] * nv[1] + u[2] * nv[2];
        const double ut = u[0] * tv[0] + u[1] * tv[1] + u[2] * tv[2];
        lit = fabs(un) <= src.sin_half2 && ua >= src.cos_half * sqrt(ua * ua + ut * ut);
    }
    if (lit) {
        double t0 = 0.0;                                 // entry parameter of the box
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            if (u[a] > 0.0) t0 = fmax(t0, (lo[a] - src.pos[a]) / u[a]);
            else if (u[a] < 0.0) t0 = fmax(t0, (lo[a] + nn[a] * del[a] - src.pos[a]) / u[a]);
        }
        int idx[3], step[3];
        double tmax[3], tdel[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            double p = src.pos[a] + t0 * u[a];
            int ii = int(floor((p - lo[a]) / del[a]));
            ii = min(max(ii, 0), nn[a] - 1);
            idx[a] = ii;
            if (u[a] > 0.0) { step[a] = 1; tmax[a] = (lo[a] + (ii + 1) * del[a] - src.pos[a]) / u[a]; tdel[a] = del[a] / u[a]; }
            else if (u[a] < 0.0) { step[a] = -1; tmax[a] = (lo[a] + ii * del[a] - src.pos[a]) / u[a]; tdel[a] = -del[a] / u[a]; }
            else { step[a] = 0; tmax[a] = INFINITY; tdel[a] = INFINITY; }
        }
        double t = t0;
        const int max_steps = m.nx + m.ny + m.nz + 4;
        for (int it = 0; it < max_steps && t < R; ++it) {
            int a = 0;
            if (tmax[1] < tmax[a]) a = 1;
            if (tmax[2] < tmax[a]) a = 2;
            double tn = fmin(tmax[a], R);
            size_t v = (size_t)idx[0] + (size_t)m.nx * (idx[1] + (size_t)m.ny * idx[2]);
            if (tn > t) sA[mat[v]][tid] += (double)rho[v] * (tn - t);
            t = tn;
            // advance along the axis that was hit (no dynamic register indexing)
            if (a == 0) { idx[0] += step[0]; tmax[0] += tdel[0]; if (idx[0] < 0 || idx[0] >= nn[0]) break; }
            else if (a == 1) { idx[1] += step[1]; tmax[1] += tdel[1]; if (idx[1] < 0 || idx[1] >= nn[1]) break; }
            else { idx[2] += step[2]; tmax[2] += tdel[2]; if (idx[2] < 0 || idx[2] >= nn[2]) break; }
        }
    }
    const double geom = 1.0 / (4.0 * 3.14159265358979323846 * R2);
    for (int g = 0; g < G; ++g) {
        double tau = 0.0;
        for (int q = 0; q < n_mat; ++q) tau += sigt_hat[q * G + g] * sA[q][tid];
        out[(size_t)g * m.cells_p] = lit ? float(spectrum[(size_t)(src0 + s) * G + g] * exp(-tau) * geom) : 0.0f;
    }
}

// sigma_t(c) = density(c) * sigt_hat[material(c)][g] for the current group, kept in fp64: the face
// recurrence of the sweep is sensitive to the rounding of sigma_t (device_common.cuh, dd_cell).
__global__ void k_sigt(MeshDev m, const uint8_t* __restrict__ mat, const float* __restrict__ rho,
                       const double* __restrict__ sigt_hat, int G, int g, double* __restrict__ sigt)
{
    long long cp = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (cp >= m.cells_p) return;
    sigt[cp] = (double)rho[cp] * sigt_hat[mat[cp] * G + g];        // padding cells carry density 0
}

// Real harmonics of reading R4 in Cartesian form (fp32), l <= 3.
template <int NM>
__device__ __forceinline__ void harmonics_f32(float mu, float eta, float xi, float* Y)
{
    Y[0] = 1.0f;
    if (NM >= 4) { Y[1] = eta; Y[2] = xi; Y[3] = mu; }
    if (NM >= 9) {
        const float s3 = 1.7320508075688772f;
        Y[4] = s3 * mu * eta; Y[5] = s3 * xi * eta; Y[6] = 0.5f * (3.0f * xi * xi - 1.0f);
        Y[7] = s3 * xi * mu;  Y[8] = 0.5f * s3 * (mu * mu - eta * eta);
    }
    if (NM >= 16) {
        const float a = 0.7905694150420949f, b = 3.872983346207417f, c = 0.6123724356957945f;
        float f = 5.0f * xi * xi - 1.0f;
        Y[9]  = a * (3.0f * mu * mu * eta - eta * eta * eta);
        Y[10] = b * xi * mu * eta;
        Y[11] = c * f * eta;
        Y[12] = 0.5f * (5.0f * xi * xi * xi - 3.0f * xi);
        Y[13] = c * f * mu;
        Y[14] = 0.5f * b * xi * (mu * mu - eta * eta);
        Y[15] = a * (mu * mu * mu - 3.0f * mu * eta * eta);
    }
}

__host__ __device__ __forceinline__ int l_of_lm(int lm) { return lm == 0 ? 0 : (lm < 4 ? 1 : (lm < 9 ? 2 : 3)); }

// =========================================================================================
// a2  Fixed source of group g (Eq. 2 right-hand side without the within-group term):
//   fixed_lm = [lm==0] S_ext^g + rho sum_{g'<=g} s_l[mat][g'->g] phi_u^{g'} Y_lm(u_c)     (Eq. 5)
//                              + rho sum_{g'<g}  s_l[mat][g'->g] phi_lm^{g'}              (downscatter)
// One thread per (cell, problem).  phi_all [prob][G][NM][cells_p], phi_u [src][G][cells_p].
// mode 0: problem p <-> source src0 + p.  mode 1: one problem, all n_src sources summed.
// =========================================================================================
template <int NM>
__global__ void __launch_bounds__(256)
k_fixed_source(MeshDev m, const uint8_t* __restrict__ mat, const float* __restrict__ rho,
               const float* __restrict__ sig_s /*[n_mat][L+1][G][G]*/, int n_mat, int L, int G, int g,
               const SourceDev* __restrict__ srcs, int src0, int n_src_members, int mode,
               const float* __restrict__ phi_u, const float* __restrict__ ext_vol /*[slot][G][cells_p]*/,
               const float* __restrict__ phi_all, float* __restrict__ fixed /*[prob][NM][cells_p]*/)
{
    extern __shared__ float s_ss[];                    // [n_mat][L+1][g+1]: s_l[mat][g' -> g]
    const int ng = g + 1;
    for (int t = threadIdx.x; t < n_mat * (L + 1) * ng; t += blockDim.x) {
        int gp = t % ng, ml = t / ng;
        s_ss[t] = sig_s[((size_t)ml * G + gp) * G + g];
    }
    __syncthreads();
    const int p = blockIdx.y;
    long long cp = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (cp >= m.cells_p) return;
    int i, j, k;
    const bool real = cell_ijk(m, cp, i, j, k);
    float* out = fixed + (size_t)p * NM * m.cells_p + cp;
    if (!real) {
#pragma unroll
        for (int lm = 0; lm < NM; ++lm) out[(size_t)lm * m.cells_p] = 0.0f;
        return;
    }
    const float dens = rho[cp];
    const float* ss = s_ss + (size_t)mat[cp] * (L + 1) * ng;
    float acc[NM];
#pragma unroll
    for (int lm = 0; lm < NM; ++lm) acc[lm] = 0.0f;

    const int s_first = mode == 0 ? src0 + p : 0;
    const int s_count = mode == 0 ? 1 : n_src_members;
    for (int sm = 0; sm < s_count; ++sm) {
        const int s = s_first + sm;                    // global source index
        const SourceDev src = srcs[s];
        if (src.kind == 0) {
            if (src.vol_slot >= 0) acc[0] += ext_vol[((size_t)src.vol_slot * G + g) * m.cells_p + cp];
            continue;
        }
        // first-collision source, Eq. (5): phi_u is a delta in angle at u_c -> moments phi_u Y_lm(u_c)
        const float* pu = phi_u + (size_t)(s - src0) * G * m.cells_p + cp;
        float ul[4] = {0.0f, 0.0f, 0.0f, 0.0f};
        for (int gp = 0; gp <= g; ++gp) {
            float v = pu[(size_t)gp * m.cells_p];
#pragma unroll
            for (int l = 0; l < 4; ++l)
                if (l <= L) ul[l] = fmaf(ss[l * ng + gp], v, ul[l]);
        }
        double ddx = m.x0 + i * m.dx - src.pos[0], ddy = m.y0 + j * m.dy - src.pos[1], ddz = m.z0 + k * m.dz - src.pos[2];
        double rinv = rsqrt(ddx * ddx + ddy * ddy + ddz * ddz);
        float Y[NM];
        harmonics_f32<NM>(float(ddx * rinv), float(ddy * rinv), float(ddz * rinv), Y);
#pragma unroll
        for (int lm = 0; lm < NM; ++lm) acc[lm] = fmaf(dens * ul[l_of_lm(lm)], Y[lm], acc[lm]);
    }
    // downscatter from the finished groups g' < g
    const float* pa = phi_all + (size_t)p * G * NM * m.cells_p + cp;
#pragma unroll 2
    for (int gp = 0; gp < g; ++gp) {                   // 2 x NM independent loads in flight per thread (streaming, HBM-bound)
        float sl[4];
#pragma unroll
        for (int l = 0; l < 4; ++l) sl[l] = l <= L ? dens * ss[l * ng + gp] : 0.0f;
#pragma unroll
        for (int lm = 0; lm < NM; ++lm)
            acc[lm] = fmaf(sl[l_of_lm(lm)], pa[((size_t)gp * NM + lm) * m.cells_p], acc[lm]);
    }
#pragma unroll
    for (int lm = 0; lm < NM; ++lm) out[(size_t)lm * m.cells_p] = acc[lm];
}

// =========================================================================================
// a6  Start of iteration k:  Q = rho s_l[mat][g->g] phi^(k-1) + fixed;  phi0_old = phi_00^(k-1);
// phi <- 0 (the sweep accumulates into it).  first = 1: phi^(0) = 0 (reading R9).
// Problems whose group already stopped are skipped.  Also resets the task counters.
// =========================================================================================
template <int NM>
__global__ void __launch_bounds__(256)
k_update(MeshDev m, const uint8_t* __restrict__ mat, const float* __restrict__ rho,
         const float* __restrict__ sig_s, int n_mat, int L, int G, int g, int Gs /*group slots in phi*/, int first,
         const float* __restrict__ fixed, float* __restrict__ phi /*[prob][Gs][NM][cells_p] at group g*/,
         float* __restrict__ Q, float* __restrict__ phi0_old, const ProbState* __restrict__ st,
         Control* ctl, double* leak)
{
    // four consecutive cells per thread: 16-byte loads and stores on every plane (cells_p is a multiple of 4: BX is)
    __shared__ float s_self[kMaxMaterials * 4];        // s_l[mat][g -> g]
    const int p = blockIdx.y;
    if (blockIdx.x == 0 && threadIdx.x < 10) {
        if (p == 0) ctl->counters[threadIdx.x] = 0u;
        if (threadIdx.x == 0 && !st[p].done) leak[p] = 0.0;
    }
    if (st[p].done) return;
    for (int t = threadIdx.x; t < n_mat * 4; t += blockDim.x) {
        const int mt = t >> 2, l = t & 3;
        s_self[t] = l <= L ? sig_s[(((size_t)mt * (L + 1) + l) * G + g) * G + g] : 0.0f;
    }
    __syncthreads();
    const long long c4 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * 4;
    if (c4 >= m.cells_p) return;
    float* ph = phi + ((size_t)p * Gs + g) * NM * m.cells_p + c4;
    float* q = Q + (size_t)p * NM * m.cells_p + c4;
    const float* fx = fixed + (size_t)p * NM * m.cells_p + c4;
    const float4 dens = *reinterpret_cast<const float4*>(rho + c4);          // padding cells: density 0, fixed 0 -> Q = 0
    const uchar4 mt = *reinterpret_cast<const uchar4*>(mat + c4);
    float4 p0 = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
#pragma unroll
    for (int lm = 0; lm < NM; ++lm) {
        const int l = l_of_lm(lm);
        const float4 f = *reinterpret_cast<const float4*>(fx + (size_t)lm * m.cells_p);
        float4 v = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        if (!first) v = *reinterpret_cast<const float4*>(ph + (size_t)lm * m.cells_p);
        if (lm == 0) p0 = v;
        float4 o;
        o.x = fmaf(dens.x * s_self[mt.x * 4 + l], v.x, f.x);
        o.y = fmaf(dens.y * s_self[mt.y * 4 + l], v.y, f.y);
        o.z = fmaf(dens.z * s_self[mt.z * 4 + l], v.z, f.z);
        o.w = fmaf(dens.w * s_self[mt.w * 4 + l], v.w, f.w);
        *reinterpret_cast<float4*>(q + (size_t)lm * m.cells_p) = o;
        *reinterpret_cast<float4*>(ph + (size_t)lm * m.cells_p) = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    }
    *reinterpret_cast<float4*>(phi0_old + (size_t)p * m.cells_p + c4) = p0;
}

// a6  End of iteration k: delta_k = max|phi_00^k - phi_00^(k-1)| / max|phi_00^k| per problem (reading R8);
// the last block to finish decides, on the device, which problems stop.
__global__ void __launch_bounds__(256)
k_check(MeshDev m, int g, int Gs, int NM, const float* __restrict__ phi, const float* __restrict__ phi0_old,
        ProbState* st, Control* ctl, int n_prob, float tol, int max_iters)
{
    const int p = blockIdx.y;
    float md = 0.0f, mp = 0.0f;
    if (!st[p].done) {
        const float* ph = phi + ((size_t)p * Gs + g) * NM * m.cells_p;
        const float* po = phi0_old + (size_t)p * m.cells_p;
        for (long long cp = (long long)blockIdx.x * blockDim.x + threadIdx.x; cp < m.cells_p;
             cp += (long long)gridDim.x * blockDim.x) {
            float v = ph[cp];
            md = fmaxf(md, fabsf(v - po[cp]));
            mp = fmaxf(mp, fabsf(v));
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        md = fmaxf(md, __shfl_xor_sync(0xffffffffu, md, o));
        mp = fmaxf(mp, __shfl_xor_sync(0xffffffffu, mp, o));
    }
    __shared__ float s_md[8], s_mp[8];
    __shared__ bool s_last;
    if ((threadIdx.x & 31) == 0) { s_md[threadIdx.x >> 5] = md; s_mp[threadIdx.x >> 5] = mp; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) { md = fmaxf(md, s_md[w]); mp = fmaxf(mp, s_mp[w]); }
        // NaN -> treat as huge so that it is visible in the residual
        if (!(md == md)) md = INFINITY;
        atomicMax(&st[p].max_diff_bits, __float_as_uint(md));
        atomicMax(&st[p].max_phi_bits, __float_as_uint(mp));
        __threadfence();
        unsigned t = atomicAdd(&ctl->ticket, 1u);
        s_last = (t == gridDim.x * gridDim.y - 1);
    }
    __syncthreads();
    if (s_last && threadIdx.x == 0) {
        __threadfence();
        int all = 1;
        for (int q = 0; q < n_prob; ++q) {
            ProbState* s = st + q;
            if (!s->done) {
                float d = __uint_as_float(atomicAdd(&s->max_diff_bits, 0u));
                float a = __uint_as_float(atomicAdd(&s->max_phi_bits, 0u));
                int k = ++s->iters;
                double delta = a == 0.0f ? 0.0 : (double)d / (double)a;
                int stop;
                if (a == 0.0f) stop = 1;                                   // no source reaches the group (R8)
                else if (s->fixed > 0) stop = k >= s->fixed;               // replay of the oracle's count (R10)
                else {
                    stop = delta < (double)tol || k >= max_iters;
                    if (!(delta < (double)tol) && k >= max_iters) s->hit_max = 1;
                }
                s->resid = (float)delta;
                s->done = stop;
                s->max_diff_bits = 0u;
                s->max_phi_bits = 0u;
            }
            all &= s->done;
        }
        ctl->all_done = all;
        ctl->ticket = 0u;
    }
}

// Balance terms of the last sweep of a group (SURVEY pins): sum Q_00 V and sum sigma_t phi_00 V, fp64.
__global__ void __launch_bounds__(256)
k_balance(MeshDev m, int g, int Gs, int NM, const float* __restrict__ phi, const float* __restrict__ Q,
          const double* __restrict__ sigt, double V, double* out /*[prob][2]*/)
{
    const int p = blockIdx.y;
    const float* ph = phi + ((size_t)p * Gs + g) * NM * m.cells_p;
    const float* q = Q + (size_t)p * NM * m.cells_p;
    double sq = 0.0, sc = 0.0;
    for (long long cp = (long long)blockIdx.x * blockDim.x + threadIdx.x; cp < m.cells_p;
         cp += (long long)gridDim.x * blockDim.x) {
        sq += (double)q[cp];
        sc += sigt[cp] * (double)ph[cp];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        sq += __shfl_xor_sync(0xffffffffu, sq, o);
        sc += __shfl_xor_sync(0xffffffffu, sc, o);
    }
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(out + 2 * p, sq * V);
        atomicAdd(out + 2 * p + 1, sc * V);
    }
}

// =========================================================================================
// sweep_mode 1 — the paper's own GPU scheme: one launch per sub-sweep S
// of one octant; thread t handles voxel cell_of[plane_offset[S] + t] (Eq. 8, Table 1 order).
// Unlike the paper, the directions of the octant are looped inside the thread, so the voxel's
// moments are reduced in registers and written once (no race on the voxel's fluence).
// Face fluxes of the octant live in global fp64 arrays out_d [prob][M][cells_p].
// =========================================================================================
template <int NM, bool FIX>
__global__ void __launch_bounds__(128)
k_subsweep(MeshDev m, const int32_t* __restrict__ cells, int count, int octant, int M,
           const float* __restrict__ Mtab, const float* __restrict__ Dtab, const double* __restrict__ dird,
           const float4* __restrict__ leakcoef,
           const double* __restrict__ sigt, const float* __restrict__ Q, float* __restrict__ phi, int g, int Gs,
           double* __restrict__ outx, double* __restrict__ outy, double* __restrict__ outz,
           const ProbState* __restrict__ st, double* leak)
{
    const int p = blockIdx.y;
    if (st[p].done) return;
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    float lk = 0.0f;
    if (t < count) {
        int c = cells[t];
        int i = c % m.nx, j = (c / m.nx) % m.ny, k = c / (m.nx * m.ny);
        size_t cp = (size_t)cell_index(m, i, j, k);
        const int sx = (octant & 1) ? -1 : 1, sy = (octant & 2) ? -1 : 1, sz = (octant & 4) ? -1 : 1;
        const int iu = i - sx, ju = j - sy, ku = k - sz;
        const bool hx = iu >= 0 && iu < m.nx, hy = ju >= 0 && ju < m.ny, hz = ku >= 0 && ku < m.nz;
        const bool bx = i + sx < 0 || i + sx >= m.nx, by = j + sy < 0 || j + sy >= m.ny, bz = k + sz < 0 || k + sz >= m.nz;
        const size_t cux = hx ? (size_t)cell_index(m, iu, j, k) : 0;
        const size_t cuy = hy ? (size_t)cell_index(m, i, ju, k) : 0;
        const size_t cuz = hz ? (size_t)cell_index(m, i, j, ku) : 0;
        const double sg = sigt[cp];
        float q[NM], acc[NM];
        const float* qp = Q + (size_t)p * NM * m.cells_p + cp;
#pragma unroll
        for (int lm = 0; lm < NM; ++lm) { q[lm] = qp[(size_t)lm * m.cells_p]; acc[lm] = 0.0f; }
        for (int n = 0; n < M; ++n) {
            const int nd = octant * M + n;
            float qn = 0.0f;
#pragma unroll
            for (int lm = 0; lm < NM; ++lm) qn = fmaf(Mtab[nd * NM + lm], q[lm], qn);
            const double dcx = dird[4 * nd], dcy = dird[4 * nd + 1], dcz = dird[4 * nd + 2], dcs = dird[4 * nd + 3];
            const size_t fo = ((size_t)p * M + n) * m.cells_p;
            double a = hx ? outx[fo + cux] : 0.0;          // vacuum inflow on the boundary
            double b = hy ? outy[fo + cuy] : 0.0;
            double cz = hz ? outz[fo + cuz] : 0.0;
            double ox, oy, oz;
            float psi = dd_cell<FIX>(true, qn, sg, dcx, dcy, dcz, dcs, a, b, cz, ox, oy, oz);
            outx[fo + cp] = ox; outy[fo + cp] = oy; outz[fo + cp] = oz;
            const float4 lc = leakcoef[nd];
            if (bx) lk = fmaf(lc.x, (float)ox, lk);
            if (by) lk = fmaf(lc.y, (float)oy, lk);
            if (bz) lk = fmaf(lc.z, (float)oz, lk);
#pragma unroll
            for (int lm = 0; lm < NM; ++lm) acc[lm] = fmaf(Dtab[nd * NM + lm], psi, acc[lm]);
        }
        float* pp = phi + ((size_t)p * Gs + g) * NM * m.cells_p + cp;
#pragma unroll
        for (int lm = 0; lm < NM; ++lm) pp[(size_t)lm * m.cells_p] += acc[lm];   // octants run one after another
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) lk += __shfl_xor_sync(0xffffffffu, lk, o);
    if ((threadIdx.x & 31) == 0 && lk != 0.0f) atomicAdd(leak + p, (double)lk);
}

// brick-major device order -> dense x-fastest [field][nz][ny][nx] (get_* calls)
__global__ void __launch_bounds__(256)
k_unbrick(MeshDev m, const float* __restrict__ src /*[fields][cells_p]*/, float* __restrict__ dst, int n_fields)
{
    const long long cells = (long long)m.nx * m.ny * m.nz;
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < cells * n_fields; c += (long long)gridDim.x * blockDim.x) {
        const int f = int(c / cells);
        const long long r = c - (long long)f * cells;
        const int i = int(r % m.nx), j = int((r / m.nx) % m.ny), kk = int(r / ((long long)m.nx * m.ny));
        dst[c] = src[(size_t)f * m.cells_p + cell_index(m, i, j, kk)];
    }
}

// Post-processing hook ("conversion of photon fluence to an absorbed dose"): a user-supplied
// response per group folded with the scalar fluence of one problem,
//   out(cell) = sum_g R_g * (phi_00,g(cell) [+ sum over the problem's sources of phi_u,s,g(cell)]),
// written dense [nz][ny][nx].  fp64 accumulation over the groups, one thread per cell, streaming reads.
__global__ void __launch_bounds__(256)
k_response(MeshDev m, int G, const double* __restrict__ resp /*[G]*/, const float* __restrict__ phi0 /*[G][cells_p] of the problem*/,
           const float* __restrict__ phiu /*[sources][G][cells_p] or NULL*/, int src0, int nsrc, float* __restrict__ dst)
{
    const long long cells = (long long)m.nx * m.ny * m.nz;
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < cells; c += (long long)gridDim.x * blockDim.x) {
        const int i = int(c % m.nx), j = int((c / m.nx) % m.ny), kk = int(c / ((long long)m.nx * m.ny));
        const long long cp = cell_index(m, i, j, kk);
        double acc = 0.0;
        for (int g = 0; g < G; ++g) {
            double f = (double)phi0[(size_t)g * m.cells_p + cp];
            if (phiu) for (int sidx = src0; sidx < src0 + nsrc; ++sidx) f += (double)phiu[((size_t)sidx * G + g) * m.cells_p + cp];
            acc = fma(resp[g], f, acc);
        }
        dst[c] = (float)acc;
    }
}

}  // namespace doctors
