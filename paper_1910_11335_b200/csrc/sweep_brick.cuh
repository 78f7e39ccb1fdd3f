// a3-a5  The product sweep kernel (sweep_mode 0): persistent CTAs sweep BRICKS of the mesh.
//
// Two-level sub-sweep schedule (Eq. 8 applied twice):
//   level 1: bricks of the brick grid; brick (bi,bj,bk) of octant o is computable once its three
//            upwind bricks are (same rule as the paper's voxels, Fig. 1).  Tasks = (problem, octant,
//            brick) are laid out in sub-sweep order of the brick grid, all 8 octants and all
//            problems interleaved, and handed out through one atomic counter; a task's upwind
//            tasks always precede it in that order, so spinning on their "done" flags cannot
//            deadlock.  No grid-wide barrier anywhere.
//   level 2: inside a brick, the cells of each i'+j'+k' = S plane (Table 1 order) are updated in
//            parallel over (cell of the plane) x (direction of the octant), __syncthreads between planes.
//
// Per task:  TMA loads Q_lm [NM][brick] and sigma_t [brick] into shared memory; phase 0 projects
// moments -> directions (q_n, a5) for the whole brick at full lane occupancy; the wavefront phase
// applies the diamond-difference update (a4) in place (q_n -> psi_n) with the three face arrays in
// shared memory; brick-to-brick faces go through small global buffers (L2 resident) guarded by
// release/acquire flags; phase 2 projects directions -> moments (Eq. 3) for the whole brick and
// one TMA reduce-add adds the tile into phi in L2 (so octants may touch a cell concurrently —
// the paper's obstacle at PAPER.md:119).  The angular flux never leaves the SM.
#pragma once
#include "device_common.cuh"

namespace doctors {

struct BrickParams {
    int nx, ny, nz;              // mesh
    int BX, BY, BZ;              // brick extents (BX % 4 == 0)
    int gbx, gby, gbz;           // brick grid
    int M;                       // directions per octant
    int g, Gs;                   // current group; group slots in the phi tensor map (coordinate 4 = prob*Gs + g)
    unsigned epoch;              // value that marks a brick done in this launch
    int task_begin, ntasks;      // slice of the task list this launch works through
    int counter_slot;
    const uint2* tasks;          // x = prob | octant << 8,  y = bi | bj << 10 | bk << 20
    Control* ctl;
    unsigned* flags;             // [prob][8][bricks]
    float* faceX;                // [prob][8][gby*gbz][M][BZ][BY]
    float* faceY;                // [prob][8][gbx*gbz][M][BZ][BX]
    float* faceZ;                // [prob][8][gbx*gby][M][BY][BX]
    const float* Mtab;           // [ndir][NM]
    const float* Dtab;           // [ndir][NM]
    const float4* dircoef;       // [ndir] {2|mu|/dx, 2|eta|/dy, 2|xi|/dz, sum}
    const float4* leakcoef;      // [ndir] {w|mu|dy dz, w|eta|dx dz, w|xi|dx dy, 0}
    const uint32_t* btab;        // in-brick schedule: i' | j' << 8 | k' << 16, BX*BY*BZ entries (Table 1 order)
    const int* bplane;           // BX+BY+BZ-1 plane offsets into btab
    const ProbState* state;
    double* leak;                // [prob]
};

__host__ __device__ inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct BrickSmem {
    size_t q, sig, psi, fx, fy, fz, dir, lk, mt, dt, tab, plane, misc, total;
};

__host__ __device__ inline BrickSmem brick_smem_layout(int NM, int BX, int BY, int BZ, int M)
{
    BrickSmem s;
    size_t NC = size_t(BX) * BY * BZ, o = 0;
    s.q = o;     o = align_up(o + NM * NC * 4, 128);
    s.sig = o;   o = align_up(o + NC * 4, 128);
    s.psi = o;   o = align_up(o + size_t(M) * NC * 4, 16);
    s.fx = o;    o = align_up(o + size_t(M) * BY * BZ * 4, 16);
    s.fy = o;    o = align_up(o + size_t(M) * BX * BZ * 4, 16);
    s.fz = o;    o = align_up(o + size_t(M) * BX * BY * 4, 16);
    s.dir = o;   o = align_up(o + size_t(M) * 16, 16);
    s.lk = o;    o = align_up(o + size_t(M) * 16, 16);
    s.mt = o;    o = align_up(o + size_t(M) * NM * 4, 16);
    s.dt = o;    o = align_up(o + size_t(M) * NM * 4, 16);
    s.tab = o;   o = align_up(o + NC * 4, 16);
    s.plane = o; o = align_up(o + size_t(BX + BY + BZ) * 4, 16);
    s.misc = o;  o = align_up(o + 64, 16);
    s.total = o;
    return s;
}

template <int NM, bool FIX>
__global__ void __launch_bounds__(kSweepThreads)
k_sweep_brick(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmPhi,
              const __grid_constant__ CUtensorMap tmSig, const BrickParams P)
{
    extern __shared__ __align__(128) unsigned char smem[];
    const int BX = P.BX, BY = P.BY, BZ = P.BZ, M = P.M;
    const int NC = BX * BY * BZ;
    const BrickSmem L = brick_smem_layout(NM, BX, BY, BZ, M);
    float* sQ = reinterpret_cast<float*>(smem + L.q);
    float* sSig = reinterpret_cast<float*>(smem + L.sig);
    float* sPsi = reinterpret_cast<float*>(smem + L.psi);
    float* sFx = reinterpret_cast<float*>(smem + L.fx);
    float* sFy = reinterpret_cast<float*>(smem + L.fy);
    float* sFz = reinterpret_cast<float*>(smem + L.fz);
    float4* sDir = reinterpret_cast<float4*>(smem + L.dir);
    float4* sLk = reinterpret_cast<float4*>(smem + L.lk);
    float* sM = reinterpret_cast<float*>(smem + L.mt);
    float* sD = reinterpret_cast<float*>(smem + L.dt);
    uint32_t* sTab = reinterpret_cast<uint32_t*>(smem + L.tab);
    int* sPlane = reinterpret_cast<int*>(smem + L.plane);
    uint64_t* sBar = reinterpret_cast<uint64_t*>(smem + L.misc);
    int* sTask = reinterpret_cast<int*>(smem + L.misc + 8);
    float* sRed = reinterpret_cast<float*>(smem + L.misc + 16);     // 8 floats

    const int tid = threadIdx.x;
    const int nplanes = BX + BY + BZ - 2;
    const uint32_t bar = smem_u32(sBar);

    // once per CTA: in-brick schedule tables, mbarrier
    for (int t = tid; t < NC; t += kSweepThreads) sTab[t] = P.btab[t];
    for (int t = tid; t <= nplanes; t += kSweepThreads) sPlane[t] = P.bplane[t];
    if (tid == 0) { mbar_init(bar, 1); fence_mbar_init(); }
    __syncthreads();
    uint32_t parity = 0;
    const int faceXn = M * BY * BZ, faceYn = M * BX * BZ, faceZn = M * BX * BY;
    const int nbricks = P.gbx * P.gby * P.gbz;

    while (true) {
        if (tid == 0) *sTask = int(atomicAdd(&P.ctl->counters[P.counter_slot], 1u));
        __syncthreads();
        const int t = *sTask;
        if (t >= P.ntasks) break;
        const uint2 td = P.tasks[P.task_begin + t];
        const int prob = td.x & 0xff, oct = (td.x >> 8) & 7;
        const int bi = td.y & 0x3ff, bj = (td.y >> 10) & 0x3ff, bk = (td.y >> 20) & 0x3ff;
        if (__ldcg(&P.state[prob].done)) { __syncthreads(); continue; }

        const int x0 = bi * BX, y0 = bj * BY, z0 = bk * BZ;
        const int ex = min(BX, P.nx - x0), ey = min(BY, P.ny - y0), ez = min(BZ, P.nz - z0);   // clipped extents
        const int sx = (oct & 1) ? -1 : 1, sy = (oct & 2) ? -1 : 1, sz = (oct & 4) ? -1 : 1;
        const bool upx = sx > 0 ? bi > 0 : bi < P.gbx - 1;
        const bool upy = sy > 0 ? bj > 0 : bj < P.gby - 1;
        const bool upz = sz > 0 ? bk > 0 : bk < P.gbz - 1;
        const bool dnx = sx > 0 ? bi < P.gbx - 1 : bi > 0;      // a downwind brick exists
        const bool dny = sy > 0 ? bj < P.gby - 1 : bj > 0;
        const bool dnz = sz > 0 ? bk < P.gbz - 1 : bk > 0;
        const int brick = bi + P.gbx * (bj + P.gby * bk);
        unsigned* flag_base = P.flags + (size_t)(prob * 8 + oct) * nbricks;
        const size_t po = (size_t)prob * 8 + oct;
        float* gFx = P.faceX + (po * (P.gby * P.gbz) + bj + P.gby * bk) * (size_t)faceXn;
        float* gFy = P.faceY + (po * (P.gbx * P.gbz) + bi + P.gbx * bk) * (size_t)faceYn;
        float* gFz = P.faceZ + (po * (P.gbx * P.gby) + bi + P.gbx * bj) * (size_t)faceZn;

        if (tid == 0) {
            bulk_wait_read0();                                   // previous tile's reduce has read sQ
            mbar_expect_tx(bar, uint32_t((NM + 1) * NC * 4));
            tma_load_5d(smem_u32(sQ), &tmQ, bar, x0, y0, z0, 0, prob);
            tma_load_3d(smem_u32(sSig), &tmSig, bar, x0, y0, z0);
            // wait for the upwind bricks of this (problem, octant)
            if (upx) while (ld_acquire_u32(flag_base + (brick - sx)) != P.epoch) __nanosleep(32);
            if (upy) while (ld_acquire_u32(flag_base + (brick - sy * P.gbx)) != P.epoch) __nanosleep(32);
            if (upz) while (ld_acquire_u32(flag_base + (brick - sz * P.gbx * P.gby)) != P.epoch) __nanosleep(32);
        }
        // octant tables (directions of this octant are contiguous: n = oct*M + m)
        for (int e = tid; e < M * NM; e += kSweepThreads) {
            sM[e] = P.Mtab[(size_t)oct * M * NM + e];
            sD[e] = P.Dtab[(size_t)oct * M * NM + e];
        }
        for (int e = tid; e < M; e += kSweepThreads) { sDir[e] = P.dircoef[oct * M + e]; sLk[e] = P.leakcoef[oct * M + e]; }
        __syncthreads();                                         // flags seen by thread 0 -> everyone may read faces

        // inflow faces: upwind brick's outflow, or vacuum
        for (int e = tid; e < faceXn; e += kSweepThreads) sFx[e] = upx ? __ldcg(gFx + e) : 0.0f;
        for (int e = tid; e < faceYn; e += kSweepThreads) sFy[e] = upy ? __ldcg(gFy + e) : 0.0f;
        for (int e = tid; e < faceZn; e += kSweepThreads) sFz[e] = upz ? __ldcg(gFz + e) : 0.0f;

        mbar_wait(bar, parity);
        parity ^= 1u;

        // ---- phase 0: q_n = sum_lm Mtab[n][lm] Q_lm for every cell of the brick (a5) ----
        for (int c0 = tid; c0 < NC; c0 += 2 * kSweepThreads) {
            const int c1 = c0 + kSweepThreads;
            const bool h1 = c1 < NC;
            float qa[NM], qb[NM];
#pragma unroll
            for (int lm = 0; lm < NM; ++lm) { qa[lm] = sQ[lm * NC + c0]; qb[lm] = h1 ? sQ[lm * NC + c1] : 0.0f; }
            for (int n = 0; n < M; ++n) {
                const float* mt = sM + n * NM;
                float a = 0.0f, b = 0.0f;
#pragma unroll
                for (int lm = 0; lm < NM; ++lm) { const float cf = mt[lm]; a = fmaf(cf, qa[lm], a); b = fmaf(cf, qb[lm], b); }
                sPsi[n * NC + c0] = a;
                if (h1) sPsi[n * NC + c1] = b;
            }
        }
        __syncthreads();

        // ---- wavefront over the i'+j'+k' = S planes of the brick (a3 level 2, a4) ----
        float lk = 0.0f;
        const bool edge_x = !dnx, edge_y = !dny, edge_z = !dnz;  // outflow faces on the mesh boundary
        for (int S = 0; S < nplanes; ++S) {
            const int beg = sPlane[S], np = sPlane[S + 1] - beg;
            const float inv_np = 1.0f / float(np);
            for (int it = tid; it < np * M; it += kSweepThreads) {
                const int n = __float2int_rz((float(it) + 0.5f) * inv_np);
                const int tt = it - n * np;
                const uint32_t e = sTab[beg + tt];
                const int ip = e & 0xff, jp = (e >> 8) & 0xff, kp = e >> 16;
                if (ip >= ex || jp >= ey || kp >= ez) continue;              // clipped brick at the mesh edge
                const int li = sx > 0 ? ip : ex - 1 - ip;
                const int lj = sy > 0 ? jp : ey - 1 - jp;
                const int lk_ = sz > 0 ? kp : ez - 1 - kp;
                const int c = li + BX * (lj + BY * lk_);
                const int ix = n * (BY * BZ) + lj + BY * lk_;
                const int iy = n * (BX * BZ) + li + BX * lk_;
                const int iz = n * (BX * BY) + li + BX * lj;
                const float4 dc = sDir[n];
                float ox, oy, oz;
                const float psi = dd_cell<FIX>(sPsi[n * NC + c], sSig[c], dc.x, dc.y, dc.z, dc.w,
                                               sFx[ix], sFy[iy], sFz[iz], ox, oy, oz);
                sPsi[n * NC + c] = psi;
                sFx[ix] = ox; sFy[iy] = oy; sFz[iz] = oz;
                if (edge_x | edge_y | edge_z) {
                    const float4 lc = sLk[n];
                    if (edge_x && ip == ex - 1) lk = fmaf(lc.x, ox, lk);
                    if (edge_y && jp == ey - 1) lk = fmaf(lc.y, oy, lk);
                    if (edge_z && kp == ez - 1) lk = fmaf(lc.z, oz, lk);
                }
            }
            __syncthreads();
        }

        // ---- outflow faces to the downwind bricks, then publish the brick ----
        if (dnx) for (int e = tid; e < faceXn; e += kSweepThreads) __stcg(gFx + e, sFx[e]);
        if (dny) for (int e = tid; e < faceYn; e += kSweepThreads) __stcg(gFy + e, sFy[e]);
        if (dnz) for (int e = tid; e < faceZn; e += kSweepThreads) __stcg(gFz + e, sFz[e]);
        if (edge_x | edge_y | edge_z) {                           // leakage through the mesh boundary
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) lk += __shfl_xor_sync(0xffffffffu, lk, o);
            if ((tid & 31) == 0) sRed[tid >> 5] = lk;
        }
        __syncthreads();
        if (tid == 0) {
            __threadfence();
            st_release_u32(flag_base + brick, P.epoch);
            if (edge_x | edge_y | edge_z) {
                float s = 0.0f;
                for (int w = 0; w < kSweepThreads / 32; ++w) s += sRed[w];
                atomicAdd(P.leak + prob, (double)s);
            }
        }

        // ---- phase 2: phi_lm += sum_n Dtab[n][lm] psi_n (Eq. 3, a5), tile -> sQ, TMA reduce-add ----
        for (int c0 = tid; c0 < NC; c0 += 2 * kSweepThreads) {
            const int c1 = c0 + kSweepThreads;
            const bool h1 = c1 < NC;
            float pa[NM], pb[NM];
#pragma unroll
            for (int lm = 0; lm < NM; ++lm) { pa[lm] = 0.0f; pb[lm] = 0.0f; }
            for (int n = 0; n < M; ++n) {
                const float* dt = sD + n * NM;
                const float va = sPsi[n * NC + c0];
                const float vb = h1 ? sPsi[n * NC + c1] : 0.0f;
#pragma unroll
                for (int lm = 0; lm < NM; ++lm) { const float cf = dt[lm]; pa[lm] = fmaf(cf, va, pa[lm]); pb[lm] = fmaf(cf, vb, pb[lm]); }
            }
#pragma unroll
            for (int lm = 0; lm < NM; ++lm) { sQ[lm * NC + c0] = pa[lm]; if (h1) sQ[lm * NC + c1] = pb[lm]; }
        }
        fence_proxy_async_smem();
        __syncthreads();
        if (tid == 0) {
            tma_reduce_add_5d(&tmPhi, smem_u32(sQ), x0, y0, z0, 0, prob * P.Gs + P.g);
            bulk_commit();
        }
    }
    if (tid == 0) bulk_wait0();
}

}  // namespace doctors
