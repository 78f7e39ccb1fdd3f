// a3-a5  The product sweep kernel (sweep_mode 0): persistent CTAs sweep BRICKS of the mesh.
//
// Two-level sub-sweep schedule (Eq. 8 applied twice):
//   level 1: bricks of the brick grid; brick (bi,bj,bk) of octant o is computable once its three
//            upwind bricks are (same rule as the paper's voxels, Fig. 1).  Tasks = (problem, octant,
//            brick) are laid out in sub-sweep order of the brick grid, all 8 octants and all
//            problems interleaved, and handed out through one atomic counter; a task's upwind
//            tasks always precede it in that order, so spinning on their "done" flags cannot
//            deadlock.  No grid-wide barrier anywhere.
//   level 2: inside a brick, ONE WARP sweeps ONE DIRECTION.  The 32 lanes are the (j',k') cross
//            section of the brick (BY x BZ <= 32) and every lane marches along x: at step s lane
//            (j',k') updates cell i' = s - j' - k', i.e. the warp's active lanes are exactly the
//            brick's cells on the paper's sub-sweep plane i'+j'+k' = s (Eq. 8).  The x face stays
//            in a register, the y and z faces are handed to lanes (j'+1,k') / (j',k'+1) by warp
//            shuffles: no shared-memory traffic, no block barrier inside the wavefront.
//
// Per task:  TMA loads Q_lm [NM][brick] (fp32) and sigma_t [brick] (fp64) into shared memory;
// phase 0 projects moments -> directions (q_n, a5) for the whole brick; the wavefront phase applies
// the diamond-difference update (a4) in place (q_n -> psi_n), its face recurrence in fp64;
// brick-to-brick faces go through global buffers (L2) guarded by release/acquire flags; phase 2
// projects directions -> moments (Eq. 3) for the whole brick and one TMA reduce-add adds the tile
// into phi in L2 (so octants may touch a cell concurrently — the paper's obstacle at PAPER.md:119).
// The angular flux never leaves the SM.
#pragma once
#include "device_common.cuh"

namespace doctors {

struct BrickParams {
    int nx, ny, nz;              // mesh
    int BX, BY, BZ;              // brick extents (BX % 4 == 0, BY * BZ <= 32)
    int gbx, gby, gbz;           // brick grid
    int M;                       // directions per octant
    int tm_rows;                 // TMA box rows per brick (tensor-map coordinate 1 of brick b = tm_rows * b)
    int W;                       // sweep warps per CTA (blockDim.x = 32 W); warp w takes directions w, w+W, ...
    int g, Gs;                   // current group; group slots in the phi tensor map (coordinate 4 = prob*Gs + g)
    unsigned epoch;              // value that marks a brick done in this launch
    int task_begin, ntasks;      // slice of the task list this launch works through
    int counter_slot;
    const uint2* tasks;          // x = prob | octant << 8,  y = bi | bj << 10 | bk << 20
    Control* ctl;
    unsigned* flags;             // [prob][8][bricks]
    double* faceX;               // [prob][8][gby*gbz][M][BZ][BY]
    double* faceY;               // [prob][8][gbx*gbz][M][BZ][BX]
    double* faceZ;               // [prob][8][gbx*gby][M][BY][BX]
    const float* Mtab;           // [ndir][NM]
    const float* Dtab;           // [ndir][NM]
    const double* dird;          // [ndir][4] {2|mu|/dx, 2|eta|/dy, 2|xi|/dz, sum}  (fp64, exact coefficients)
    const float4* leakcoef;      // [ndir] {w|mu|dy dz, w|eta|dx dz, w|xi|dx dy, 0}
    const ProbState* state;
    double* leak;                // [prob]
    int bulk_faces;              // 1: all three face blocks are multiples of 16 bytes -> moved by bulk async copies (TMA unit)
    long long* dbg_time;         // -DDOCTORS_TIMING builds only: [16] cycle sums per phase (thread 0 of every CTA)
    int* dbg_plane;              // debug hook: NULL, or [BX*BY*BZ] receives the step at which each cell of a full brick is visited
};

__host__ __device__ inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct BrickSmem {
    size_t q, sig, psi, fx, fy, fz, dir, lk, mt, dt, misc, total;
};

__host__ __device__ inline BrickSmem brick_smem_layout(int NM, int BX, int BY, int BZ, int M)
{
    BrickSmem s;
    size_t NC = size_t(BX) * BY * BZ, o = 0;
    s.misc = o;  o = align_up(o + 128, 128);   // mbarrier, task slots, reduction scratch; also the pad idle lanes may read
    // one tile of max(NM, M) planes holds, in turn, Q_lm (TMA load), psi_n (in place, per cell) and the
    // phi_lm contribution (in place again, TMA reduce-add source)
    s.q = o;     o = align_up(o + size_t(NM > M ? NM : M) * NC * 4, 128);
    s.sig = o;   o = align_up(o + NC * 8, 128);
    s.psi = s.q;
    s.fx = o;    o = align_up(o + size_t(M) * BY * BZ * 8, 8);      // fx, fy, fz contiguous (one load loop)
    s.fy = o;    o = align_up(o + size_t(M) * BX * BZ * 8, 8);
    s.fz = o;    o = align_up(o + size_t(M) * BX * BY * 8, 16);
    s.dir = o;   o = align_up(o + size_t(M) * 32, 16);
    s.lk = o;    o = align_up(o + size_t(M) * 16, 16);
    s.mt = o;    o = align_up(o + size_t(M) * ((NM + 3) / 4 * 4) * 4, 16);
    s.dt = o;    o = align_up(o + size_t(M) * ((NM + 3) / 4 * 4) * 4, 16);
    o = align_up(o + 128, 16);                  // tail pad (idle lanes may read up to 10 cells past the tables' start)
    s.total = o;
    return s;
}

// Sub-sweep indexing inside a brick (Eq. 8): lane -> (j',k') of the cross section, step s -> i'.
__device__ __forceinline__ void lane_cross_section(int lane, int BY, int& jp, int& kp)
{
    jp = lane % BY;
    kp = lane / BY;
}
constexpr int kFaceRegs = 7;
template <int NM> __host__ __device__ constexpr int kTabPitch() { return (NM + 3) / 4 * 4; }   // table row pitch (16-byte rows)
__device__ __forceinline__ int step_to_ip(int s, int jp, int kp) { return s - jp - kp; }

template <int NM, bool FIX, bool DBG = false>
__global__ void __launch_bounds__(32 * kMaxSweepWarps, 3)
k_sweep_brick(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmPhi,
              const __grid_constant__ CUtensorMap tmSig, const BrickParams P)
{
    if (__ldcg(&P.ctl->all_done)) return;                              // every problem of the chunk has stopped (a6): nothing to sweep
    extern __shared__ __align__(128) unsigned char smem[];
    const int BX = P.BX, BY = P.BY, BZ = P.BZ, M = P.M;
    const int NC = BX * BY * BZ;
    const BrickSmem L = brick_smem_layout(NM, BX, BY, BZ, M);
    float* sQ = reinterpret_cast<float*>(smem + L.q);
    double* sSig = reinterpret_cast<double*>(smem + L.sig);
    float* sPsi = reinterpret_cast<float*>(smem + L.psi);
    double* sFx = reinterpret_cast<double*>(smem + L.fx);
    double* sFy = reinterpret_cast<double*>(smem + L.fy);
    double* sFz = reinterpret_cast<double*>(smem + L.fz);
    double* sDir = reinterpret_cast<double*>(smem + L.dir);          // [M][4]
    float4* sLk = reinterpret_cast<float4*>(smem + L.lk);
    float* sM = reinterpret_cast<float*>(smem + L.mt);
    float* sD = reinterpret_cast<float*>(smem + L.dt);
    uint64_t* sBar = reinterpret_cast<uint64_t*>(smem + L.misc);
    int* sTask = reinterpret_cast<int*>(smem + L.misc + 8);
    float* sRed = reinterpret_cast<float*>(smem + L.misc + 64);     // kMaxSweepWarps floats

    const int tid = threadIdx.x, nthr = blockDim.x;
    const int lane = tid & 31, warp = tid >> 5;
    const uint32_t bar = smem_u32(sBar);
    int jp, kp;
    lane_cross_section(lane, BY, jp, kp);

    const uint32_t barF = bar + 32;                                  // faces (bulk copies) complete here
    if (tid == 0) { mbar_init(bar, 1); mbar_init(barF, 1); fence_mbar_init(); }
    __syncthreads();
    uint32_t parity = 0;
    const int faceXn = M * BY * BZ, faceYn = M * BX * BZ, faceZn = M * BX * BY;
    const int nbricks = P.gbx * P.gby * P.gbz;
    int last_oct = -1;
#ifdef DOCTORS_TIMING
    long long tacc[12] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}, tprev = clock64();
#define TICK(i) do { if (tid == 0) { long long t_ = clock64(); tacc[i] += t_ - tprev; tprev = t_; } } while (0)
#else
#define TICK(i) do { } while (0)
#endif

    // The id of the next task is fetched one task ahead (the atomic's round trip hides behind the
    // sweep).  Holding one unstarted task cannot deadlock: a CTA's held task has a higher index than
    // its running one, so the lowest unfinished task of the whole grid is always running.
    if (tid == 0) sTask[0] = int(atomicAdd(&P.ctl->counters[P.counter_slot], 1u));
    int slot = 0;
    while (true) {
        __syncthreads();
        const int t = sTask[slot];
        if (t >= P.ntasks) break;
        if (tid == 32 % nthr) sTask[slot ^ 1] = int(atomicAdd(&P.ctl->counters[P.counter_slot], 1u));
        slot ^= 1;
        TICK(0);
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
        double* gFx = P.faceX + (po * (P.gby * P.gbz) + bj + P.gby * bk) * (size_t)faceXn;
        double* gFy = P.faceY + (po * (P.gbx * P.gbz) + bi + P.gbx * bk) * (size_t)faceYn;
        double* gFz = P.faceZ + (po * (P.gbx * P.gby) + bi + P.gbx * bj) * (size_t)faceZn;

        // octant tables (directions of this octant are contiguous: n = oct*M + m): loaded by warps 1.. while
        // warp 0 issues the tile load and polls the flags, so that their global-load latency is hidden
        if (oct != last_oct) {
            const int tt = nthr > 32 ? tid - 32 : tid, tn = nthr > 32 ? nthr - 32 : nthr;
            if (tt >= 0) {
                for (int e = tt; e < M * NM; e += tn) {
                    const int n = e / NM, lm = e - n * NM;
                    sM[n * kTabPitch<NM>() + lm] = P.Mtab[(size_t)oct * M * NM + e];
                    sD[n * kTabPitch<NM>() + lm] = P.Dtab[(size_t)oct * M * NM + e];
                }
                for (int e = tt; e < M * 4; e += tn) sDir[e] = P.dird[(size_t)oct * M * 4 + e];
                for (int e = tt; e < M; e += tn) sLk[e] = P.leakcoef[oct * M + e];
            }
            last_oct = oct;
        }
        if (tid == 0) {
            bulk_wait_read0();                                   // previous tile's reduce has read sQ
            mbar_expect_tx(bar, uint32_t(NM * NC * 4 + NC * 8));
            tma_load_4d(smem_u32(sQ), &tmQ, bar, 0, P.tm_rows * brick, 0, prob);
            tma_load_2d(smem_u32(sSig), &tmSig, bar, 0, P.tm_rows * brick);
        }
        TICK(9);
        // wait for the upwind bricks of this (problem, octant): one warp-0 lane per upwind flag
        if (warp == 0) {
            const bool need = lane == 0 ? upx : (lane == 1 ? upy : (lane == 2 && upz));
            const int up = lane == 0 ? brick - sx : (lane == 1 ? brick - sy * P.gbx : brick - sz * P.gbx * P.gby);
            bool ready = !need;
            while (!__all_sync(0xffffffffu, ready)) {
                if (!ready) ready = ld_acquire_u32(flag_base + up) == P.epoch;
            }
        }
        TICK(10);
        __syncthreads();                                         // flags seen by thread 0 -> everyone may read faces
        TICK(1);

        // inflow faces: upwind brick's outflow, or vacuum.  sFx, sFy, sFz are contiguous.
        const int nxy = faceXn + faceYn, nall = nxy + faceZn;
        double fv[kFaceRegs];
        if (P.bulk_faces) {
            // one thread hands the three blocks to the TMA unit (1-D bulk copies, complete on barF);
            // vacuum faces are zero-filled by the threads.  Nothing here waits: the data is needed after phase 0.
            if (tid == 0) {
                fence_proxy_async_all();                         // flags acquired (generic proxy) -> async-proxy reads
                mbar_expect_tx(barF, uint32_t(8 * ((upx ? faceXn : 0) + (upy ? faceYn : 0) + (upz ? faceZn : 0))));
                if (upx) bulk_load(smem_u32(sFx), gFx, uint32_t(8 * faceXn), barF);
                if (upy) bulk_load(smem_u32(sFy), gFy, uint32_t(8 * faceYn), barF);
                if (upz) bulk_load(smem_u32(sFz), gFz, uint32_t(8 * faceZn), barF);
            }
            if (!upx) for (int e = tid; e < faceXn; e += nthr) sFx[e] = 0.0;
            if (!upy) for (int e = tid; e < faceYn; e += nthr) sFy[e] = 0.0;
            if (!upz) for (int e = tid; e < faceZn; e += nthr) sFz[e] = 0.0;
        } else {
            // odd-sized blocks: the first kFaceRegs elements of every thread travel through registers (their
            // loads are issued here and parked in shared memory after phase 0), the rest is copied directly
#pragma unroll
            for (int k = 0; k < kFaceRegs; ++k) {
                const int e = tid + k * nthr;
                const double* src = e < faceXn ? gFx + e : (e < nxy ? gFy + (e - faceXn) : gFz + (e - nxy));
                const bool u = e < faceXn ? upx : (e < nxy ? upy : upz);
                fv[k] = (e < nall && u) ? __ldcg(src) : 0.0;
            }
            for (int e = tid + kFaceRegs * nthr; e < nall; e += nthr) {
                const double* src = e < faceXn ? gFx + e : (e < nxy ? gFy + (e - faceXn) : gFz + (e - nxy));
                const bool u = e < faceXn ? upx : (e < nxy ? upy : upz);
                sFx[e] = u ? __ldcg(src) : 0.0;
            }
        }
        TICK(2);
        mbar_wait(bar, parity);
        parity ^= 1u;
        TICK(3);

        // ---- phase 0: q_n = sum_lm Mtab[n][lm] Q_lm for every cell of the brick (a5) ----
        // Two cells per thread share every coefficient load (the phase is bound by the shared-memory pipe);
        // packed fp32x2 FMAs (FFMA2, sm_100) accumulate even / odd moments in the halves of a register pair.
        for (int c = tid; c < NC; c += 2 * nthr) {
            const int c2 = c + nthr;
            const bool two = c2 < NC;
            if constexpr (NM >= 2) {
                float2 qa[NM / 2], qb[NM / 2];
#pragma unroll
                for (int k = 0; k < NM / 2; ++k) {
                    qa[k] = make_float2(sQ[(2 * k) * NC + c], sQ[(2 * k + 1) * NC + c]);
                    qb[k] = two ? make_float2(sQ[(2 * k) * NC + c2], sQ[(2 * k + 1) * NC + c2]) : make_float2(0.0f, 0.0f);
                }
                float qla = 0.0f, qlb = 0.0f;
                if (NM & 1) { qla = sQ[(NM - 1) * NC + c]; qlb = two ? sQ[(NM - 1) * NC + c2] : 0.0f; }
                for (int n = 0; n < M; ++n) {
                    const float2* mt = reinterpret_cast<const float2*>(sM + n * kTabPitch<NM>());
                    float2 a = make_float2(0.0f, 0.0f), b = make_float2(0.0f, 0.0f);
#pragma unroll
                    for (int k = 0; k < NM / 2; ++k) { const float2 m2 = mt[k]; a = __ffma2_rn(m2, qa[k], a); b = __ffma2_rn(m2, qb[k], b); }
                    float ra = a.x + a.y, rb = b.x + b.y;
                    if (NM & 1) { const float ml = sM[n * kTabPitch<NM>() + NM - 1]; ra = fmaf(ml, qla, ra); rb = fmaf(ml, qlb, rb); }
                    sPsi[n * NC + c] = ra;                       // in place: this thread has read all of its cells
                    if (two) sPsi[n * NC + c2] = rb;
                }
            } else {
                const float qa0 = sQ[c], qb0 = two ? sQ[c2] : 0.0f;
                for (int n = 0; n < M; ++n) {
                    const float m0 = sM[n * kTabPitch<NM>()];
                    sPsi[n * NC + c] = m0 * qa0;
                    if (two) sPsi[n * NC + c2] = m0 * qb0;
                }
            }
        }
        if (P.bulk_faces) {
            mbar_wait(barF, parity ^ 1u);                         // same phase sequence as `bar` (flipped above)
        } else {
#pragma unroll
            for (int k = 0; k < kFaceRegs; ++k) {
                const int e = tid + k * nthr;
                if (e < nall) sFx[e] = fv[k];
            }
        }
        __syncthreads();
        TICK(4);

        // ---- wavefront (a3 level 2, a4): warp = direction, lanes = (j',k'), step s -> plane i'+j'+k' = s ----
        const bool edge_x = !dnx, edge_y = !dny, edge_z = !dnz;  // outflow faces on the mesh boundary
        const bool lane_ok = kp < ez && jp < ey;
        const int lj = sy > 0 ? jp : ey - 1 - jp;
        const int lk_ = sz > 0 ? kp : ez - 1 - kp;
        const int nsteps = ex + ey + ez - 2;
        const bool last_y = jp == ey - 1, last_z = kp == ez - 1;
        const int li0 = (sx > 0 ? 0 : ex - 1) - sx * (jp + kp);   // li at step 0 (i' = -(j'+k')), advanced by sx per step
        const uint32_t row = uint32_t(BX * (lj + BY * lk_) + li0);
        const bool first_y = jp == 0, first_z = kp == 0;
        // Idle lanes (before / after their x range) load from wherever their running address points — always
        // inside this CTA's shared memory, which starts with a 128-byte pad and ends with the tables — and
        // compute on that garbage; only stores and the x-face register are predicated.  Clipped lanes
        // (beyond ey / ez) stay parked on the tile's first cell.
        const int d4 = lane_ok ? 4 * sx : 0, d8 = 2 * d4;
        const int shy = BY;
        for (int n = warp; n < M; n += P.W) {
            const double cx = sDir[4 * n], cy = sDir[4 * n + 1], cz = sDir[4 * n + 2], cs = sDir[4 * n + 3];
            double* fxp = sFx + n * (BY * BZ) + lj + BY * lk_;
            // running shared-memory addresses of this lane's cell: advanced by one cell (sx) per step
            uint32_t pq = smem_u32(sPsi) + (lane_ok ? 4u * (uint32_t(n * NC) + row) : 0u);
            uint32_t ps = smem_u32(sSig) + (lane_ok ? 8u * row : 0u);
            uint32_t py = smem_u32(sFy) + (lane_ok ? 8u * uint32_t((n * BZ + lk_) * BX + li0) : 0u);
            uint32_t pz = smem_u32(sFz) + (lane_ok ? 8u * uint32_t((n * BY + lj) * BX + li0) : 0u);
            double ax = lane_ok ? *fxp : 0.0, oy = 0.0, oz = 0.0;
            int ip = lane_ok ? -(jp + kp) : -(1 << 29);          // clipped lanes never become active
#pragma unroll 1
            for (int s = nsteps; s > 0; --s) {
                double b = __shfl_up_sync(0xffffffffu, oy, 1);
                double cc = __shfl_up_sync(0xffffffffu, oz, shy);
                const bool act = (unsigned)ip < (unsigned)ex;    // this lane's cell lies on the current sub-sweep plane
                const float q = lds_f32(pq);
                const double sg = lds_f64(ps);
                if (first_y) b = lds_f64(py);
                if (first_z) cc = lds_f64(pz);
                double ox;
                const float psi = dd_cell<FIX>(act, q, sg, cx, cy, cz, cs, ax, b, cc, ox, oy, oz);
                sts_f32_if(act, pq, psi);
                sts_f64_if(act && last_y, py, oy);
                sts_f64_if(act && last_z, pz, oz);
                if (act) ax = ox;
                if (DBG && act) P.dbg_plane[(pq - smem_u32(sPsi)) / 4u - uint32_t(n * NC)] = nsteps - s;
                ++ip; pq += d4; ps += d8; py += d8; pz += d8;
            }
            if (lane_ok) *fxp = ax;
        }
        __syncthreads();
        TICK(5);

        // leakage through the mesh boundary (balance report): sum of w |Omega_d| A_d psi_out over boundary faces
        if (edge_x | edge_y | edge_z) {
            float lk = 0.0f;
            if (edge_x) for (int e = tid; e < faceXn; e += nthr) {
                const int n = e / (BY * BZ), r = e - n * (BY * BZ);
                if (r % BY < ey && r / BY < ez) lk = fmaf(sLk[n].x, (float)sFx[e], lk);
            }
            if (edge_y) for (int e = tid; e < faceYn; e += nthr) {
                const int n = e / (BX * BZ), r = e - n * (BX * BZ);
                if (r % BX < ex && r / BX < ez) lk = fmaf(sLk[n].y, (float)sFy[e], lk);
            }
            if (edge_z) for (int e = tid; e < faceZn; e += nthr) {
                const int n = e / (BX * BY), r = e - n * (BX * BY);
                if (r % BX < ex && r / BX < ey) lk = fmaf(sLk[n].z, (float)sFz[e], lk);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) lk += __shfl_xor_sync(0xffffffffu, lk, o);
            if (lane == 0) sRed[warp] = lk;
        }

        // ---- outflow faces to the downwind bricks, then publish the brick ----
        if (P.bulk_faces) {
            fence_proxy_async_smem();                            // lanes' face writes -> visible to the async proxy
            __syncthreads();
            if (tid == nthr - 1) {
                if (dnx) bulk_store(gFx, smem_u32(sFx), uint32_t(8 * faceXn));
                if (dny) bulk_store(gFy, smem_u32(sFy), uint32_t(8 * faceYn));
                if (dnz) bulk_store(gFz, smem_u32(sFz), uint32_t(8 * faceZn));
                bulk_commit();
            }
        } else {
            if (dnx) for (int e = tid; e < faceXn; e += nthr) __stcg(gFx + e, sFx[e]);
            if (dny) for (int e = tid; e < faceYn; e += nthr) __stcg(gFy + e, sFy[e]);
            if (dnz) for (int e = tid; e < faceZn; e += nthr) __stcg(gFz + e, sFz[e]);
            __syncthreads();
            if (tid == nthr - 1) st_release_u32(flag_base + brick, P.epoch);   // cumulative: covers the CTA's face stores (ordered by the barrier)
        }
        TICK(6);

        // ---- phase 2: phi_lm += sum_n Dtab[n][lm] psi_n (Eq. 3, a5), tile -> sQ, TMA reduce-add ----
        for (int c = tid; c < NC; c += 2 * nthr) {
            const int c2 = c + nthr;
            const bool two = c2 < NC;
            if constexpr (NM >= 2) {
                float2 pa[NM / 2], pb[NM / 2];
                float pla = 0.0f, plb = 0.0f;
#pragma unroll
                for (int k = 0; k < NM / 2; ++k) { pa[k] = make_float2(0.0f, 0.0f); pb[k] = make_float2(0.0f, 0.0f); }
                for (int n = 0; n < M; ++n) {
                    const float2* dt = reinterpret_cast<const float2*>(sD + n * kTabPitch<NM>());
                    const float va = sPsi[n * NC + c], vb = two ? sPsi[n * NC + c2] : 0.0f;
                    const float2 va2 = make_float2(va, va), vb2 = make_float2(vb, vb);
#pragma unroll
                    for (int k = 0; k < NM / 2; ++k) { const float2 d2 = dt[k]; pa[k] = __ffma2_rn(d2, va2, pa[k]); pb[k] = __ffma2_rn(d2, vb2, pb[k]); }
                    if (NM & 1) { const float dl = sD[n * kTabPitch<NM>() + NM - 1]; pla = fmaf(dl, va, pla); plb = fmaf(dl, vb, plb); }
                }
#pragma unroll
                for (int k = 0; k < NM / 2; ++k) {
                    sQ[(2 * k) * NC + c] = pa[k].x; sQ[(2 * k + 1) * NC + c] = pa[k].y;
                    if (two) { sQ[(2 * k) * NC + c2] = pb[k].x; sQ[(2 * k + 1) * NC + c2] = pb[k].y; }
                }
                if (NM & 1) { sQ[(NM - 1) * NC + c] = pla; if (two) sQ[(NM - 1) * NC + c2] = plb; }
            } else {
                float pa0 = 0.0f, pb0 = 0.0f;
                for (int n = 0; n < M; ++n) {
                    const float d0 = sD[n * kTabPitch<NM>()];
                    pa0 = fmaf(d0, sPsi[n * NC + c], pa0);
                    if (two) pb0 = fmaf(d0, sPsi[n * NC + c2], pb0);
                }
                sQ[c] = pa0;
                if (two) sQ[c2] = pb0;
            }
        }
        fence_proxy_async_smem();
        __syncthreads();
        TICK(7);
        if (P.bulk_faces && tid == nthr - 1) {                   // publish the brick; the others already start the next task
            bulk_wait0();                                        // face blocks are in global memory (and read out of sFx..sFz)
            fence_proxy_async_all();
            st_release_u32(flag_base + brick, P.epoch);
        }
        if (tid == 0) {
            tma_reduce_add_4d(&tmPhi, smem_u32(sQ), 0, P.tm_rows * brick, 0, prob * P.Gs + P.g);
            bulk_commit();
            if (edge_x | edge_y | edge_z) {
                float s = 0.0f;
                for (int w = 0; w < P.W; ++w) s += sRed[w];
                atomicAdd(P.leak + prob, (double)s);
            }
        }
    }
    if (tid == 0) bulk_wait0();
#ifdef DOCTORS_TIMING
    if (tid == 0 && P.dbg_time) {
        tacc[8] = clock64() - tprev;
        for (int i = 0; i < 12; ++i) atomicAdd(reinterpret_cast<unsigned long long*>(P.dbg_time) + i, (unsigned long long)tacc[i]);
    }
#endif
#undef TICK
}

}  // namespace doctors
