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
// Per task:  one tensor copy (TMA, 4-D box) brings the dense tile Q_lm [NM][brick] (fp32) into shared memory — with the
// tensor-core projections, whose planes are padded, one 1-D bulk copy per moment plane instead —, 1-D bulk copies bring
// sigma_t [brick] (fp64) and, when the CTA changes octant, the octant's table blob; phase 0 projects moments ->
// directions (q_n, a5) for the whole brick; the wavefront phase applies the diamond-difference update (a4) in place
// (q_n -> psi_n), its face recurrence in fp64; brick-to-brick faces (fp32 with closure 1, fp64 with closure 0: FaceOf) go through global buffers guarded by
// release/acquire flags; phase 2 projects directions -> moments (Eq. 3) for the whole brick and one tensor reduce-add
// (cp.reduce.async.bulk.tensor .add.f32) adds the tile into phi in L2 (so octants may touch a cell concurrently — the
// paper's obstacle at PAPER.md:119).  The angular flux never leaves the SM.
//
// Projections (a5), template parameter MT:
//   MT = 0  plain FFMA2 loops (any NM, any M).
//   MT >= 1 (NM = 16, M <= 16 MT): the two 16-wide contractions run on the tensor cores as
//           mma.sync m16n8k8 TF32 with the 3-product split (a_hi b_lo + a_lo b_hi + a_hi b_hi, fp32
//           accumulate): per-term relative error ~2^-21, well inside the 1e-4 gate.  The
//           coefficient tables arrive pre-split and in fragment order (host_tables / api.cu), moment planes
//           sit at a pitch = 8 (mod 32) words so fragment loads and stores are bank-conflict free.
#pragma once
#include "device_common.cuh"

namespace doctors {

// Storage type of the faces EXCHANGED between bricks (global buffers and the shared-memory face arrays of a task).  The
// recurrence inside a brick is fp64 (registers, shuffles) either way; only what crosses a brick boundary is stored: every
// 20th x face, 8th y face and 4th z face of a ray.
//   closure 1 (FIX, the gated closure of configs 2-4): fp32.  Halves the only DRAM traffic in excess of the algorithmic bytes
//     (1.32 x -> 1.17 x) and 11 KB of shared memory per CTA; the whole config-4 solve stays within 3.8e-6 of the oracle
//     (1.2e-6 with fp64 faces), and the power it saves lifts the power-capped SM clock of the whole solve from ~1865 to 1950 MHz.
//   closure 0 (pure diamond difference): fp64.  Its ill-conditioned cells (sign changes of phi_0 in the lowest groups) lose
//     with fp32 exchange faces: 24 instead of 3-4 of 202722 stored cells of config 4 above 1e-4.
template <bool FIX> struct FaceOf { using type = double; };
template <> struct FaceOf<true> { using type = float; };
__host__ __device__ constexpr unsigned face_bytes(bool fix) { return fix ? 4u : 8u; }
template <typename F>
__device__ __forceinline__ double load_face(uint32_t a)
{
    if constexpr (sizeof(F) == 8) return lds_f64(a); else return (double)lds_f32(a);
}
template <typename F>
__device__ __forceinline__ void store_face_if(bool p, uint32_t a, double v)
{
    if constexpr (sizeof(F) == 8) sts_f64_if(p, a, v); else sts_f32_if(p, a, (float)v);
}

struct BrickParams {
    int nx, ny, nz;              // mesh
    int BX, BY, BZ;              // brick extents (BX % 4 == 0, BY * BZ <= 32)
    int gbx, gby, gbz;           // brick grid
    int M;                       // directions per octant
    int nprob;                   // problems the task list refers to (<= 256)
    int NCb;                     // cells per brick (= BX*BY*BZ): brick b of a per-cell array starts at b * NCb
    int tm_rows;                 // tensor maps of Q / phi: a brick = tm_rows box rows (coordinate 1 of brick b = tm_rows * b)
    long long cells_p;           // padded cell count (plane pitch of Q / phi in global memory)
    const float* Q;              // [prob][NM][cells_p]
    float* phi;                  // [prob * Gs + g][NM][cells_p]
    const double* sigt;          // [cells_p], current group
    const unsigned char* octtab; // [8] blobs of octtab_layout(...).total bytes
    int W;                       // sweep warps per CTA (blockDim.x = 32 W); warp w takes directions w, w+W, ...
    int g, Gs;                   // current group; group slots in the phi tensor map (coordinate 4 = prob*Gs + g)
    unsigned epoch;              // value that marks a brick done in this launch
    int task_begin, ntasks;      // slice of the task list this launch works through
    int counter_slot;
    const uint2* tasks;          // x = prob | octant << 8,  y = bi | bj << 10 | bk << 20
    Control* ctl;
    unsigned* flags;             // [prob][8][bricks]
    void* faceX;                 // [prob][8][gby*gbz][M][BZ][BY]   float (closure 1) or double (closure 0), see FaceOf
    void* faceY;                 // [prob][8][gbx*gbz][M][BZ][BX]
    void* faceZ;                 // [prob][8][gbx*gby][M][BY][BX]
    const ProbState* state;
    double* leak;                // [prob]
    int bulk_faces;              // 1: all three face blocks are multiples of 16 bytes -> moved by bulk async copies (TMA unit)
    int* dbg_plane;              // debug hook: NULL, or [BX*BY*BZ + 1]: the step at which each cell of a full brick is visited,
                                 // then the count of out-of-allocation shared-memory addresses of the wavefront loop
};

__host__ __device__ inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

constexpr int kFragBytes = 512;   // one mma A fragment (4 x b32) for the 32 lanes of a warp
template <int NM> __host__ __device__ constexpr int kTabPitch() { return (NM + 3) / 4 * 4; }   // table row pitch (16-byte rows)

// Per-octant table blob (global memory, copied to shared memory by one bulk copy when a CTA changes octant):
//   dir  [M][4] double  {2|mu|/dx, 2|eta|/dy, 2|xi|/dz, sum}   (fp64, exact coefficients)
//   lk   [M] float4     {w|mu|dy dz, w|eta|dx dz, w|xi|dx dy, 0}
//   MT = 0:  mt [M][pitch], dt [M][pitch] float  (moment -> direction, direction -> moment)
//   MT >= 1: a0 [MT][2 k-steps][hi, lo][32 lanes] float4: A fragments of Mtab (rows = directions, K = moments)
//            a2 [2 MT k-steps][hi, lo][32 lanes] float4: A fragments of Dtab^T (rows = moments, K = directions, zero beyond M)
struct OctTab { size_t dir, lk, t0, t2, total; };
__host__ __device__ inline OctTab octtab_layout(int NM, int M, int MT)
{
    OctTab o;
    const size_t pitch = size_t((NM + 3) / 4 * 4);
    o.dir = 0;
    o.lk = size_t(M) * 32;
    o.t0 = o.lk + size_t(M) * 16;
    if (MT == 0) { o.t2 = o.t0 + size_t(M) * pitch * 4; o.total = o.t2 + size_t(M) * pitch * 4; }
    else { o.t2 = o.t0 + size_t(MT) * 2 * 2 * kFragBytes; o.total = o.t2 + size_t(2 * MT) * 2 * kFragBytes; }
    o.total = (o.total + 15) / 16 * 16;
    return o;
}

// plane pitch (in floats) of the moment / direction tile in shared memory
__host__ __device__ inline int plane_pitch(int NC, int MT)
{
    if (MT == 0) return NC;
    return NC + (8 - NC % 32 + 32) % 32;       // = 8 (mod 32): conflict-free mma fragment loads / stores
}

struct BrickSmem {
    size_t q, sig, psi, fx, fy, fz, tab, done, misc, total;
};

__host__ __device__ inline BrickSmem brick_smem_layout(int NM, int BX, int BY, int BZ, int M, int MT, unsigned kFaceBytes)
{
    BrickSmem s;
    size_t NC = size_t(BX) * BY * BZ, o = 0;
    s.misc = o;  o = align_up(o + 256, 128);   // mbarriers, reduction scratch, two decoded task slots (TaskSlot) at +128
    // front pad: a wavefront lane that has not reached its x range yet loads from its running address, up to
    // (BY + BZ - 2) steps of BY cells (8 bytes each for sigma_t) BEFORE its row — that must still be this CTA's memory
    o = align_up(o + size_t(8) * BY * (BY + BZ - 2), 128);
    // one tile of max(NM, M) planes holds, in turn, Q_lm (bulk loads), psi_n (in place, per cell) and the
    // phi_lm contribution (in place again, bulk reduce-add source)
    s.q = o;     o = align_up(o + size_t(NM > M ? NM : M) * plane_pitch(int(NC), MT) * 4, 128);
    s.sig = o;   o = align_up(o + NC * 8, 128);
    s.psi = s.q;
    s.fx = o;    o = align_up(o + size_t(M) * BY * BZ * kFaceBytes, kFaceBytes);      // fx, fy, fz contiguous (one load loop)
    s.fy = o;    o = align_up(o + size_t(M) * BX * BZ * kFaceBytes, kFaceBytes);
    s.fz = o;    o = align_up(o + size_t(M) * BX * BY * kFaceBytes, 16);
    s.tab = o;   o = align_up(o + octtab_layout(NM, M, MT).total, 16);
    s.done = o;  o = align_up(o + 256, 16);      // "problem has stopped" bytes of the launch (task prob index is 8 bits)
    o = align_up(o + 128 + size_t(8) * BY * (BY + BZ - 2), 16);   // tail pad: lanes past their x range (sx < 0: before it) overshoot by the same amount
    s.total = o;
    return s;
}

// m-tiles of 16 directions the tensor-core projections need; 0 = use the FFMA2 loops
__host__ __device__ inline int projection_mtiles(int NM, int M, int NC)
{
    if (NM != 16 || NC % 8 != 0 || M > 48) return 0;
    return (M + 15) / 16;
}

// Sub-sweep indexing inside a brick (Eq. 8): lane -> (j',k') of the cross section, step s -> i'.
__device__ __forceinline__ void lane_cross_section(int lane, int BY, int& jp, int& kp)
{
    jp = lane % BY;
    kp = lane / BY;
}
constexpr int kFaceRegs = 7;
__device__ __forceinline__ int step_to_ip(int s, int jp, int kp) { return s - jp - kp; }

// ---- a5 on the tensor cores ------------------------------------------------------------------------------
// Both projections are [16 x K] x [K x cells] contractions with K <= 48.  One n-tile = 8 consecutive cells of the
// brick; a warp works on two n-tiles at a time and reads every plane of those cells before it writes the result
// over the same planes (in place).  Each (tile, k-step) pair owns an accumulator: four independent chains of
// three dependent MMAs, issued round-robin in source order (ptxas keeps mma.sync in program order; a dependent
// HMMA waits ~21 cycles, an independent one issues every 8 — measured on B200).
// Kept out of line: the kernel around them is register-starved (64 registers for 3 CTAs per SM) and these
// loops want their own allocation; the call costs a few spills per task instead of rematerialised addresses
// in every iteration.
struct MmaChains {
    float acc[2][2][4];                                       // [tile][k-step]
    __device__ __forceinline__ void clear()
    {
#pragma unroll
        for (int u = 0; u < 2; ++u)
#pragma unroll
            for (int k = 0; k < 2; ++k) { acc[u][k][0] = 0.0f; acc[u][k][1] = 0.0f; acc[u][k][2] = 0.0f; acc[u][k][3] = 0.0f; }
    }
    // acc[u][k] += A_k * B_{u,k} with the 3-product TF32 split; small terms first
    __device__ __forceinline__ void run(const float4 (&ah)[2], const float4 (&al)[2], const float (&bh)[2][4], const float (&bl)[2][4])
    {
#pragma unroll
        for (int k = 0; k < 2; ++k)
#pragma unroll
            for (int u = 0; u < 2; ++u) mma_tf32(acc[u][k], al[k], bh[u][2 * k], bh[u][2 * k + 1]);
#pragma unroll
        for (int k = 0; k < 2; ++k)
#pragma unroll
            for (int u = 0; u < 2; ++u) mma_tf32(acc[u][k], ah[k], bl[u][2 * k], bl[u][2 * k + 1]);
#pragma unroll
        for (int k = 0; k < 2; ++k)
#pragma unroll
            for (int u = 0; u < 2; ++u) mma_tf32(acc[u][k], ah[k], bh[u][2 * k], bh[u][2 * k + 1]);
    }
};

// moments -> directions:  q_n[cell] = sum_lm Mtab[n][lm] Q_lm[cell]   (rhs of Eq. 2 in moment form, R3)
// `tile`: shared address of plane 0, `frag`: shared address of the a0 fragments (octtab_layout)
template <int MT>
__device__ __noinline__ void project_moments_to_directions_mma(uint32_t tile, uint32_t frag, int NC, int NCP, int M)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int gq = lane >> 2, tq = lane & 3;
    const int NT = NC >> 3;
    const uint32_t p4 = 16u * uint32_t(NCP);                  // four planes, in bytes
    const uint32_t ld0 = tile + 4u * uint32_t(tq * NCP + gq);
    const uint32_t st0 = tile + 4u * uint32_t(gq * NCP + 2 * tq);
    const uint32_t fl = frag + 16u * uint32_t(lane);
    float4 ah[2], al[2];
    if constexpr (MT == 1) {
#pragma unroll
        for (int ks = 0; ks < 2; ++ks) { ah[ks] = lds_v4f32(fl + uint32_t(ks * 2 + 0) * kFragBytes); al[ks] = lds_v4f32(fl + uint32_t(ks * 2 + 1) * kFragBytes); }
    }
#pragma unroll 1
    for (int t0 = 2 * warp; t0 < NT; t0 += 2 * nwarps) {
        const bool two = t0 + 1 < NT;                          // a missing second tile recomputes the first (not stored)
        float bh[2][4], bl[2][4];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const uint32_t a = ld0 + 32u * uint32_t(t0 + (two ? u : 0));
#pragma unroll
            for (int r = 0; r < 4; ++r) split_tf32(lds_f32(a + uint32_t(r) * p4), bh[u][r], bl[u][r]);   // lm = tq + 4 r
        }
        float out[MT][2][4];
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) {
            if constexpr (MT > 1) {
#pragma unroll
                for (int ks = 0; ks < 2; ++ks) { ah[ks] = lds_v4f32(fl + uint32_t((mt * 2 + ks) * 2 + 0) * kFragBytes); al[ks] = lds_v4f32(fl + uint32_t((mt * 2 + ks) * 2 + 1) * kFragBytes); }
            }
            MmaChains C;
            C.clear();
            C.run(ah, al, bh, bl);
#pragma unroll
            for (int u = 0; u < 2; ++u)
#pragma unroll
                for (int e = 0; e < 4; ++e) out[mt][u][e] = C.acc[u][0][e] + C.acc[u][1][e];
        }
        __syncwarp();
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            if (u == 0 || two) {
                const uint32_t d = st0 + 32u * uint32_t(t0 + u);
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    const int n0 = 16 * mt + gq;
                    if (n0 < M) sts_v2f32(d + uint32_t(4 * mt) * p4, out[mt][u][0], out[mt][u][1]);
                    if (n0 + 8 < M) sts_v2f32(d + uint32_t(4 * mt + 2) * p4, out[mt][u][2], out[mt][u][3]);
                }
            }
        }
    }
}

// directions -> moments:  phi_lm[cell] (this octant's share) = sum_n Dtab[n][lm] psi_n[cell]   (Eq. 3)
// K = 16 MT directions, two 8-wide k-steps per pass; the fragments are zero beyond M and those planes are not read.
template <int MT>
__device__ __noinline__ void project_directions_to_moments_mma(uint32_t tile, uint32_t frag, int NC, int NCP, int M)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int gq = lane >> 2, tq = lane & 3;
    const int NT = NC >> 3;
    const uint32_t p4 = 16u * uint32_t(NCP);
    const uint32_t ld0 = tile + 4u * uint32_t(tq * NCP + gq);
    const uint32_t st0 = tile + 4u * uint32_t(gq * NCP + 2 * tq);
    const uint32_t fl = frag + 16u * uint32_t(lane);
    float4 ah[2], al[2];
    if constexpr (MT == 1) {
#pragma unroll
        for (int ks = 0; ks < 2; ++ks) { ah[ks] = lds_v4f32(fl + uint32_t(ks * 2 + 0) * kFragBytes); al[ks] = lds_v4f32(fl + uint32_t(ks * 2 + 1) * kFragBytes); }
    }
#pragma unroll 1
    for (int t0 = 2 * warp; t0 < NT; t0 += 2 * nwarps) {
        const bool two = t0 + 1 < NT;
        MmaChains C;
        C.clear();
#pragma unroll
        for (int kp = 0; kp < MT; ++kp) {                     // pass kp: directions 16 kp .. 16 kp + 15
            if (16 * kp < M) {                                // uniform
                if constexpr (MT > 1) {
#pragma unroll
                    for (int ks = 0; ks < 2; ++ks) { ah[ks] = lds_v4f32(fl + uint32_t((kp * 2 + ks) * 2 + 0) * kFragBytes); al[ks] = lds_v4f32(fl + uint32_t((kp * 2 + ks) * 2 + 1) * kFragBytes); }
                }
                float bh[2][4], bl[2][4];
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    const uint32_t a = ld0 + 32u * uint32_t(t0 + (two ? u : 0)) + uint32_t(4 * kp) * p4;
#pragma unroll
                    for (int r = 0; r < 4; ++r) {             // direction n = 16 kp + tq + 4 r  (k-step r / 2)
                        const float v = 16 * kp + tq + 4 * r < M ? lds_f32(a + uint32_t(r) * p4) : 0.0f;
                        split_tf32(v, bh[u][r], bl[u][r]);
                    }
                }
                C.run(ah, al, bh, bl);
            }
        }
        __syncwarp();
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            if (u == 0 || two) {
                const uint32_t d = st0 + 32u * uint32_t(t0 + u);
                sts_v2f32(d, C.acc[u][0][0] + C.acc[u][1][0], C.acc[u][0][1] + C.acc[u][1][1]);
                sts_v2f32(d + 2u * p4, C.acc[u][0][2] + C.acc[u][1][2], C.acc[u][0][3] + C.acc[u][1][3]);
            }
        }
    }
}

// A task as the sweeping warps consume it: decoded ONCE by the thread that fetches it (while the previous task runs) instead of
// by every warp of the CTA (the decode was ~100 instructions per warp and task, 8 % of all instructions executed: profiles/).
struct __align__(16) TaskSlot {
    int id;                        // position in the task list (>= ntasks: no more work)
    unsigned bits;                 // prob | oct << 8 | upx, upy, upz, dnx, dny, dnz << 16.. | stopped << 24
    int brick;
    unsigned ext;                  // clipped extents ex | ey << 8 | ez << 16
    unsigned long long gFx, gFy, gFz;   // this brick's face blocks in the global exchange buffers
    unsigned long long flag_base;       // done-flags of (prob, oct): [bricks]
    unsigned long long pad;
};
static_assert(sizeof(TaskSlot) == 64, "two slots fit the misc area");

// PITCH > 0: the brick holds exactly PITCH cells (the default 20 x 8 x 4 = 640) and the plane pitch of the tile is a compile-time
// constant: the 32 plane addresses a thread touches in each projection become immediates off one base register (they were an
// IMAD each), and the octant has 10 directions (S8: the projection loops have a constant trip count).  PITCH = 0: any brick and
// quadrature, from the parameters.  The brick's EXTENTS and the thread count stay run-time values either way (as constants they
// cost more in spills at the 64-register cap than they save: measured 8.59 against 8.31 ms).
template <int NM, bool FIX, int MT, int PITCH, bool DBG = false>
__global__ void __launch_bounds__(32 * kMaxSweepWarps, 3)
k_sweep_brick(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmPhi, const BrickParams P)
{
    static_assert(MT == 0 || NM == 16, "tensor-core projections are written for P3 (16 moments)");
    static_assert(NM <= 16, "one tile-warp lane per moment plane, lanes 16 / 17 for sigma_t and the tables");
    if (__ldcg(&P.ctl->all_done)) return;                              // every problem of the chunk has stopped (a6): nothing to sweep
    extern __shared__ __align__(128) unsigned char smem[];
    const int BX = P.BX, BY = P.BY, BZ = P.BZ, M = PITCH ? 10 : P.M;   // fixed pitch: S8, 10 directions per octant
    static_assert(PITCH == 0 || MT == 0, "a fixed pitch is instantiated for the dense (FMA-loop) tile only");
    const int NC = PITCH ? PITCH : BX * BY * BZ;
    const int NCP = PITCH ? PITCH : plane_pitch(NC, MT);              // plane pitch of the tile (floats)
    using face_t = typename FaceOf<FIX>::type;
    constexpr unsigned kFaceBytes = sizeof(face_t);
    const BrickSmem L = brick_smem_layout(NM, BX, BY, BZ, M, MT, kFaceBytes);
    const OctTab T = octtab_layout(NM, M, MT);
    float* sQ = reinterpret_cast<float*>(smem + L.q);
    double* sSig = reinterpret_cast<double*>(smem + L.sig);
    float* sPsi = reinterpret_cast<float*>(smem + L.psi);
    face_t* sFx = reinterpret_cast<face_t*>(smem + L.fx);
    face_t* sFy = reinterpret_cast<face_t*>(smem + L.fy);
    face_t* sFz = reinterpret_cast<face_t*>(smem + L.fz);
    double* sDir = reinterpret_cast<double*>(smem + L.tab + T.dir);  // [M][4]
    float4* sLk = reinterpret_cast<float4*>(smem + L.tab + T.lk);
    float* sM = reinterpret_cast<float*>(smem + L.tab + T.t0);      // MT = 0: [M][pitch];  MT >= 1: A fragments (float4 per lane)
    float* sD = reinterpret_cast<float*>(smem + L.tab + T.t2);
    uint64_t* sBar = reinterpret_cast<uint64_t*>(smem + L.misc);
    float* sRed = reinterpret_cast<float*>(smem + L.misc + 64);     // kMaxSweepWarps floats

    const int tid = threadIdx.x, nthr = blockDim.x;
    const int lane = tid & 31, warp = tid >> 5;
    const uint32_t bar = smem_u32(sBar);
    int jp, kp;
    lane_cross_section(lane, BY, jp, kp);

    const uint32_t barF = bar + 32;                                  // faces (bulk copies) complete here
    if (tid == 0) { mbar_init(bar, 1); mbar_init(barF, P.bulk_faces ? 3 : 1); fence_mbar_init(); }
    uint32_t parity = 0;
    const int faceXn = M * BY * BZ, faceYn = M * BX * BZ, faceZn = M * BX * BY;
    const int nbricks = P.gbx * P.gby * P.gbz;
    int last_oct = -1;

    // Roles inside the CTA (all of them also sweep):
    //   tile warp   lanes 0..NM-1 own one moment plane each: bulk load of Q_lm at the start of a task, bulk reduce-add of
    //               the phi_lm contribution at its end (same lane = same bulk group, so the lane can wait for "read done")
    //   pollers     warp 0, lanes 0..2: wait for the upwind brick in x / y / z and issue that face's bulk load themselves
    //   prefetcher  one thread fetches the NEXT task (id from the atomic counter, then its descriptor) into shared memory
    //               while the current one runs: two dependent global round trips off the critical path.
    //               Holding one unstarted task cannot deadlock: a CTA's held task has a higher index than its running one,
    //               so the lowest unfinished task of the whole grid is always running.
    //   publisher   last lane of the last warp: bulk-stores the outflow faces, and at the next loop top waits for them and
    //               releases the brick's flag AFTER arriving at the block barrier (split barrier: nobody waits for it)
    const int nwarps = nthr >> 5;
    const int tileWarp = nwarps > 1 ? 1 : 0;
    const int pfThread = nwarps > 2 ? 64 : 32 * tileWarp + 8;
    const int pubWarp = nwarps - 1;
    TaskSlot* sSlot = reinterpret_cast<TaskSlot*>(smem + L.misc + 128);   // [2]
    unsigned char* sDoneP = smem + L.done;                        // [nprob]: fixed for the whole launch (k_check runs between launches)
    for (int q = tid; q < P.nprob; q += nthr) sDoneP[q] = (unsigned char)(__ldcg(&P.state[q].done) != 0);
    auto fetch_task = [&](int sl) {
        const int id = int(atomicAdd(&P.ctl->counters[P.counter_slot], 1u));
        TaskSlot t;
        t.id = id; t.bits = 0u; t.brick = 0; t.ext = 0u; t.gFx = t.gFy = t.gFz = t.flag_base = t.pad = 0ull;
        if (id < P.ntasks) {
            const uint2 d = P.tasks[P.task_begin + id];
            const int prob = d.x & 0xff, oct = (d.x >> 8) & 7;
            const int bi = d.y & 0x3ff, bj = (d.y >> 10) & 0x3ff, bk = (d.y >> 20) & 0x3ff;
            const int ex = min(BX, P.nx - bi * BX), ey = min(BY, P.ny - bj * BY), ez = min(BZ, P.nz - bk * BZ);   // clipped extents
            const bool px = !(oct & 1), py_ = !(oct & 2), pz_ = !(oct & 4);
            const unsigned upx = px ? bi > 0 : bi < P.gbx - 1, upy = py_ ? bj > 0 : bj < P.gby - 1, upz = pz_ ? bk > 0 : bk < P.gbz - 1;
            const unsigned dnx = px ? bi < P.gbx - 1 : bi > 0, dny = py_ ? bj < P.gby - 1 : bj > 0, dnz = pz_ ? bk < P.gbz - 1 : bk > 0;
            t.bits = unsigned(prob) | unsigned(oct) << 8 | upx << 16 | upy << 17 | upz << 18 | dnx << 19 | dny << 20 | dnz << 21 |
                     unsigned(sDoneP[prob]) << 24;
            t.brick = bi + P.gbx * (bj + P.gby * bk);
            t.ext = unsigned(ex) | unsigned(ey) << 8 | unsigned(ez) << 16;
            const size_t po = (size_t)prob * 8 + oct;
            t.gFx = reinterpret_cast<unsigned long long>(static_cast<face_t*>(P.faceX) + (po * (P.gby * P.gbz) + bj + P.gby * bk) * (size_t)faceXn);
            t.gFy = reinterpret_cast<unsigned long long>(static_cast<face_t*>(P.faceY) + (po * (P.gbx * P.gbz) + bi + P.gbx * bk) * (size_t)faceYn);
            t.gFz = reinterpret_cast<unsigned long long>(static_cast<face_t*>(P.faceZ) + (po * (P.gbx * P.gby) + bi + P.gbx * bj) * (size_t)faceZn);
            t.flag_base = reinterpret_cast<unsigned long long>(P.flags + po * (size_t)nbricks);
        }
        sSlot[sl] = t;
    };
    __syncthreads();                                             // stop flags (read by fetch_task)
    if (tid == 0) fetch_task(0);
    __syncthreads();                                             // mbarriers, first task
    int slot = 0;
    // ONE block barrier ends a task (after phase 2): behind it nobody reads the tile, the tables, the faces or the task
    // slot of that task any more, so the next task starts without a barrier of its own.
    while (true) {
        const TaskSlot& ts = sSlot[slot];
        const int t = ts.id;
        if (t >= P.ntasks) break;
        const unsigned tb = ts.bits;
        if (tid == pfThread) fetch_task(slot ^ 1);
        slot ^= 1;
        if (tb >> 24) { __syncthreads(); continue; }             // this problem has stopped (a6); the barrier orders the task slots
        const int prob = tb & 0xff, oct = (tb >> 8) & 7;
        const unsigned te = ts.ext;
        const int ex = te & 0xff, ey = (te >> 8) & 0xff, ez = te >> 16;
        const int sx = (oct & 1) ? -1 : 1, sy = (oct & 2) ? -1 : 1, sz = (oct & 4) ? -1 : 1;
        const bool upx = (tb >> 16) & 1, upy = (tb >> 17) & 1, upz = (tb >> 18) & 1;
        const bool dnx = (tb >> 19) & 1, dny = (tb >> 20) & 1, dnz = (tb >> 21) & 1;      // a downwind brick exists
        const int brick = ts.brick;
        unsigned* flag_base = reinterpret_cast<unsigned*>(ts.flag_base);
        face_t* gFx = reinterpret_cast<face_t*>(ts.gFx);
        face_t* gFy = reinterpret_cast<face_t*>(ts.gFy);
        face_t* gFz = reinterpret_cast<face_t*>(ts.gFz);

        // tile, sigma_t and (when the octant changes) the octant's table blob: bulk async copies, one mbarrier.
        // Directions of an octant are contiguous (n = oct*M + m); nobody reads the old tables any more (loop-top barrier).
        if (warp == tileWarp) {
            const bool tab = oct != last_oct;
            if (lane == 0) mbar_expect_tx(bar, uint32_t(NM * NC * 4 + NC * 8 + (tab ? T.total : 0)));
            const float* gq = P.Q + (size_t)prob * NM * P.cells_p + (size_t)brick * P.NCb;
            if constexpr (MT == 0) {
                // dense tile [NM][brick]: ONE tensor copy (4-D box {row, rows of the brick, moments, problem}); issuing a bulk
                // operation costs ~200 cycles of the issuing warp, so one per moment plane is only used where the planes
                // are padded in shared memory (tensor-core projections)
                if (lane == 0) {
                    bulk_wait_read0();                           // the reduce-add of the previous task has read the tile
                    tma_load_4d(smem_u32(sQ), &tmQ, bar, 0, P.tm_rows * brick, 0, prob);
                }
            } else if (lane < NM) {
                bulk_wait_read0();                               // this lane's reduce-add of the previous task has read its plane
                bulk_load(smem_u32(sQ + lane * NCP), gq + (size_t)lane * P.cells_p, uint32_t(NC * 4), bar);
            }
            if (lane == 16) bulk_load(smem_u32(sSig), P.sigt + (size_t)brick * P.NCb, uint32_t(NC * 8), bar);
            if (tab && lane == 17) bulk_load(smem_u32(smem + L.tab), P.octtab + (size_t)oct * T.total, uint32_t(T.total), bar);
        }
        last_oct = oct;
        // wait for the upwind bricks of this (problem, octant): one warp-0 lane per upwind flag
        if (P.bulk_faces) {
            if (warp == 0 && lane < 3) {
                const bool need = lane == 0 ? upx : (lane == 1 ? upy : upz);
                if (need) {
                    const int up = lane == 0 ? brick - sx : (lane == 1 ? brick - sy * P.gbx : brick - sz * P.gbx * P.gby);
                    const face_t* src = lane == 0 ? gFx : (lane == 1 ? gFy : gFz);
                    const uint32_t dst = smem_u32(lane == 0 ? sFx : (lane == 1 ? sFy : sFz));
                    const uint32_t bytes = kFaceBytes * uint32_t(lane == 0 ? faceXn : (lane == 1 ? faceYn : faceZn));
                    while (ld_acquire_u32(flag_base + up) != P.epoch) { }
                    fence_proxy_async_global();                     // flag acquired (generic proxy) -> async-proxy read of the face
                    mbar_expect_tx(barF, bytes);
                    bulk_load(dst, src, bytes, barF);            // 1-D bulk copy (TMA unit); needed after phase 0
                } else {
                    mbar_arrive(barF);
                }
            }
        } else {
            if (warp == 0) {
                const bool need = lane == 0 ? upx : (lane == 1 ? upy : (lane == 2 && upz));
                const int up = lane == 0 ? brick - sx : (lane == 1 ? brick - sy * P.gbx : brick - sz * P.gbx * P.gby);
                bool ready = !need;
                while (!__all_sync(0xffffffffu, ready)) {
                    if (!ready) ready = ld_acquire_u32(flag_base + up) == P.epoch;
                }
            }
            __syncthreads();                                     // flags seen by warp 0 -> everyone may read faces
        }

        // inflow faces: upwind brick's outflow, or vacuum.  sFx, sFy, sFz are contiguous.
        const int nxy = faceXn + faceYn, nall = nxy + faceZn;
        face_t fv[kFaceRegs];
        if (P.bulk_faces) {
            // vacuum faces are zero-filled by the threads; the others arrive by the pollers' bulk copies
            if (!upx) for (int e = tid; e < faceXn; e += nthr) sFx[e] = face_t(0);
            if (!upy) for (int e = tid; e < faceYn; e += nthr) sFy[e] = face_t(0);
            if (!upz) for (int e = tid; e < faceZn; e += nthr) sFz[e] = face_t(0);
        } else {
            // odd-sized blocks: the first kFaceRegs elements of every thread travel through registers (their
            // loads are issued here and parked in shared memory after phase 0), the rest is copied directly
#pragma unroll
            for (int k = 0; k < kFaceRegs; ++k) {
                const int e = tid + k * nthr;
                const face_t* src = e < faceXn ? gFx + e : (e < nxy ? gFy + (e - faceXn) : gFz + (e - nxy));
                const bool u = e < faceXn ? upx : (e < nxy ? upy : upz);
                fv[k] = (e < nall && u) ? __ldcg(src) : face_t(0);
            }
            for (int e = tid + kFaceRegs * nthr; e < nall; e += nthr) {
                const face_t* src = e < faceXn ? gFx + e : (e < nxy ? gFy + (e - faceXn) : gFz + (e - nxy));
                const bool u = e < faceXn ? upx : (e < nxy ? upy : upz);
                sFx[e] = u ? __ldcg(src) : face_t(0);
            }
        }
        mbar_wait(bar, parity);
        parity ^= 1u;

        // ---- phase 0: q_n = sum_lm Mtab[n][lm] Q_lm for every cell of the brick (a5) ----
        if constexpr (MT >= 1) {
            project_moments_to_directions_mma<MT>(smem_u32(sQ), smem_u32(sM), NC, NCP, M);
        } else {
            // Two cells per thread share every coefficient load (the phase is bound by the shared-memory pipe);
            // packed fp32x2 FMAs (FFMA2, sm_100) accumulate even / odd moments in the halves of a register pair.
            // two cells per thread, (c, c + NC/2): NC is even (BX is a multiple of 4), so every thread of every round has both,
            // whatever the brick length (768 cells on 320 threads: one round of 320 pairs, one of 64)
            for (int c = tid; c < NC / 2; c += nthr) {
                const int c2 = c + NC / 2;
                constexpr bool two = true;
                if constexpr (NM >= 2) {
                    float2 qa[NM / 2], qb[NM / 2];
    #pragma unroll
                    for (int k = 0; k < NM / 2; ++k) {
                        qa[k] = make_float2(sQ[(2 * k) * NCP + c], sQ[(2 * k + 1) * NCP + c]);
                        qb[k] = two ? make_float2(sQ[(2 * k) * NCP + c2], sQ[(2 * k + 1) * NCP + c2]) : make_float2(0.0f, 0.0f);
                    }
                    float qla = 0.0f, qlb = 0.0f;
                    if (NM & 1) { qla = sQ[(NM - 1) * NCP + c]; qlb = two ? sQ[(NM - 1) * NCP + c2] : 0.0f; }
                    for (int n = 0; n < M; ++n) {
                        const float2* mt = reinterpret_cast<const float2*>(sM + n * kTabPitch<NM>());
                        float2 a = make_float2(0.0f, 0.0f), b = make_float2(0.0f, 0.0f);
    #pragma unroll
                        for (int k = 0; k < NM / 2; ++k) { const float2 m2 = mt[k]; a = __ffma2_rn(m2, qa[k], a); b = __ffma2_rn(m2, qb[k], b); }
                        float ra = a.x + a.y, rb = b.x + b.y;
                        if (NM & 1) { const float ml = sM[n * kTabPitch<NM>() + NM - 1]; ra = fmaf(ml, qla, ra); rb = fmaf(ml, qlb, rb); }
                        sPsi[n * NCP + c] = ra;                       // in place: this thread has read all of its cells
                        if (two) sPsi[n * NCP + c2] = rb;
                    }
                } else {
                    const float qa0 = sQ[c], qb0 = two ? sQ[c2] : 0.0f;
                    for (int n = 0; n < M; ++n) {
                        const float m0 = sM[n * kTabPitch<NM>()];
                        sPsi[n * NCP + c] = m0 * qa0;
                        if (two) sPsi[n * NCP + c2] = m0 * qb0;
                    }
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

        // ---- wavefront (a3 level 2, a4): warp = direction, lanes = (j',k'), step s -> plane i'+j'+k' = s ----
        const bool edge_x = !dnx, edge_y = !dny, edge_z = !dnz;  // outflow faces on the mesh boundary
        const bool lane_ok = kp < ez && jp < ey;
        const int lj = sy > 0 ? jp : ey - 1 - jp;
        const int lk_ = sz > 0 ? kp : ez - 1 - kp;
        const int nsteps = ex + ey + ez - 2;
        const bool last_y = jp == ey - 1, last_z = kp == ez - 1;
        const int li0 = (sx > 0 ? 0 : ex - 1) - sx * (jp + kp);   // li at step 0 (i' = -(j'+k')), advanced by sx per step
        const uint32_t row = uint32_t(lj + BY * (li0 + BX * lk_));    // local index: y fastest, then x, then z (device_common.cuh)
        const bool first_y = jp == 0, first_z = kp == 0;
        // Idle lanes (before / after their x range) keep advancing their running addresses but touch nothing (masked below); the
        // pads in front of and behind the tile keep even those addresses inside this CTA's shared memory (the debug
        // instantiation checks that).  Clipped lanes (beyond ey / ez) stay parked on the tile's first cell.
        int d4 = lane_ok ? 4 * sx * BY : 0, d8 = 2 * d4, d8f = lane_ok ? int(kFaceBytes) * sx : 0;   // one cell along x: tile (fp32), sigma_t (fp64), face rows
        int shy = BY, ly = last_y ? 1 : 0, lz = last_z ? 1 : 0;
        // loop invariants pinned in registers: otherwise the compiler re-derives them every step (constant-bank reads,
        // ey - 1 / ez - 1 on the uniform datapath, 2 * d4)
        asm volatile("" : "+r"(d4), "+r"(d8), "+r"(d8f), "+r"(shy), "+r"(ly), "+r"(lz));
        for (int n = warp; n < M; n += P.W) {
            const double cx = sDir[4 * n], cy = sDir[4 * n + 1], cz = sDir[4 * n + 2], cs = sDir[4 * n + 3];
            face_t* fxp = sFx + n * (BY * BZ) + lj + BY * lk_;
            // running shared-memory addresses of this lane's cell: advanced by one cell (sx) per step
            uint32_t pq = smem_u32(sPsi) + (lane_ok ? 4u * (uint32_t(n * NCP) + row) : 0u);
            uint32_t ps = smem_u32(sSig) + (lane_ok ? 8u * row : 0u);
            uint32_t py = smem_u32(sFy) + (lane_ok ? kFaceBytes * uint32_t((n * BZ + lk_) * BX + li0) : 0u);
            uint32_t pz = smem_u32(sFz) + (lane_ok ? kFaceBytes * uint32_t((n * BY + lj) * BX + li0) : 0u);
            double ax = lane_ok ? (double)*fxp : 0.0, oy = 0.0, oz = 0.0;
            int ip = lane_ok ? -(jp + kp) : -(1 << 29);          // clipped lanes never become active
#pragma unroll 1
            for (int s = nsteps; s > 0; --s) {
                double b = __shfl_up_sync(0xffffffffu, oy, 1);
                double cc = __shfl_up_sync(0xffffffffu, oz, shy);
                const bool act = (unsigned)ip < (unsigned)ex;    // this lane's cell lies on the current sub-sweep plane
                // Lanes outside their x range are masked off (a divergent branch, not predicated garbage arithmetic).  At equal
                // clock that costs 1 % (8.36 against 8.27 ms per slice launch), but the whole solve runs under the 1000 W cap and a
                // third of the lane-steps are idle: masked, the SM clock settles at 1927 instead of 1878 MHz and the solve is 1.2 %
                // faster (profiles/r02_sweep_ncu.md).  The shuffles above stay outside: every lane takes part in them.
                if (act) {
                    const float q = lds_f32(pq);
                    const double sg = lds_f64(ps);
                    if (first_y) b = load_face<face_t>(py);
                    if (first_z) cc = load_face<face_t>(pz);
                    double ox;
                    const float psi = dd_cell<FIX>(true, q, sg, cx, cy, cz, cs, ax, b, cc, ox, oy, oz);
                    sts_f32(pq, psi);
                    store_face_if<face_t>(ly, py, oy);
                    store_face_if<face_t>(lz, pz, oz);
                    ax = ox;
                }
                if (DBG) {
                    // debug instantiation (doctors_debug_device_brick_steps): the step at which each cell is visited, and a
                    // bounds check of EVERY shared-memory address of the step, idle lanes included (they load from their
                    // running addresses, see above): slot NC of dbg_plane counts addresses outside this CTA's allocation
                    if (act) P.dbg_plane[(pq - smem_u32(sPsi)) / 4u - uint32_t(n * NCP)] = nsteps - s;   // indexed by the storage order (y fastest)
                    const uint32_t lo = smem_u32(smem), hi = lo + uint32_t(L.total);
                    const bool bad = pq < lo || pq + 4u > hi || ps < lo || ps + 8u > hi || py < lo || py + kFaceBytes > hi || pz < lo || pz + kFaceBytes > hi;
                    if (bad) atomicAdd(P.dbg_plane + NC, 1);
                }
                ++ip; pq += d4; ps += d8; py += d8f; pz += d8f;
            }
            if (lane_ok) *fxp = face_t(ax);
        }
        if (P.bulk_faces) fence_proxy_async_smem();              // lanes' face writes -> visible to the async proxy
        __syncthreads();
        // ---- outflow faces to the downwind bricks: bulk async stores issued by the publisher (last lane of the last warp) ----
        if (P.bulk_faces && warp == pubWarp && lane == 31) {
            if (dnx) bulk_store(gFx, smem_u32(sFx), uint32_t(kFaceBytes * faceXn));
            if (dny) bulk_store(gFy, smem_u32(sFy), uint32_t(kFaceBytes * faceYn));
            if (dnz) bulk_store(gFz, smem_u32(sFz), uint32_t(kFaceBytes * faceZn));
            bulk_commit();
        }

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

        if (!P.bulk_faces) {                                     // odd-sized face blocks: plain stores, flag after a barrier
            if (dnx) for (int e = tid; e < faceXn; e += nthr) __stcg(gFx + e, sFx[e]);
            if (dny) for (int e = tid; e < faceYn; e += nthr) __stcg(gFy + e, sFy[e]);
            if (dnz) for (int e = tid; e < faceZn; e += nthr) __stcg(gFz + e, sFz[e]);
            __syncthreads();
            if (tid == nthr - 1) st_release_u32(flag_base + brick, P.epoch);   // cumulative: covers the CTA's face stores (ordered by the barrier)
        }

        // ---- phase 2: phi_lm += sum_n Dtab[n][lm] psi_n (Eq. 3, a5), tile -> sQ, bulk reduce-adds ----
        if constexpr (MT >= 1) {
            project_directions_to_moments_mma<MT>(smem_u32(sQ), smem_u32(sD), NC, NCP, M);
        } else {
            // two cells per thread, (c, c + NC/2): NC is even (BX is a multiple of 4), so every thread of every round has both,
            // whatever the brick length (768 cells on 320 threads: one round of 320 pairs, one of 64)
            for (int c = tid; c < NC / 2; c += nthr) {
                const int c2 = c + NC / 2;
                constexpr bool two = true;
                if constexpr (NM >= 2) {
                    float2 pa[NM / 2], pb[NM / 2];
                    float pla = 0.0f, plb = 0.0f;
    #pragma unroll
                    for (int k = 0; k < NM / 2; ++k) { pa[k] = make_float2(0.0f, 0.0f); pb[k] = make_float2(0.0f, 0.0f); }
                    for (int n = 0; n < M; ++n) {
                        const float2* dt = reinterpret_cast<const float2*>(sD + n * kTabPitch<NM>());
                        const float va = sPsi[n * NCP + c], vb = two ? sPsi[n * NCP + c2] : 0.0f;
                        const float2 va2 = make_float2(va, va), vb2 = make_float2(vb, vb);
    #pragma unroll
                        for (int k = 0; k < NM / 2; ++k) { const float2 d2 = dt[k]; pa[k] = __ffma2_rn(d2, va2, pa[k]); pb[k] = __ffma2_rn(d2, vb2, pb[k]); }
                        if (NM & 1) { const float dl = sD[n * kTabPitch<NM>() + NM - 1]; pla = fmaf(dl, va, pla); plb = fmaf(dl, vb, plb); }
                    }
    #pragma unroll
                    for (int k = 0; k < NM / 2; ++k) {
                        sQ[(2 * k) * NCP + c] = pa[k].x; sQ[(2 * k + 1) * NCP + c] = pa[k].y;
                        if (two) { sQ[(2 * k) * NCP + c2] = pb[k].x; sQ[(2 * k + 1) * NCP + c2] = pb[k].y; }
                    }
                    if (NM & 1) { sQ[(NM - 1) * NCP + c] = pla; if (two) sQ[(NM - 1) * NCP + c2] = plb; }
                } else {
                    float pa0 = 0.0f, pb0 = 0.0f;
                    for (int n = 0; n < M; ++n) {
                        const float d0 = sD[n * kTabPitch<NM>()];
                        pa0 = fmaf(d0, sPsi[n * NCP + c], pa0);
                        if (two) pb0 = fmaf(d0, sPsi[n * NCP + c2], pb0);
                    }
                    sQ[c] = pa0;
                    if (two) sQ[c2] = pb0;
                }
            }
        }
        const bool publisher = P.bulk_faces && warp == pubWarp && lane == 31;
        if (publisher) bulk_wait_read0();                        // the face blocks have been read out of sFx..sFz (issued before phase 2)
        fence_proxy_async_smem();
        __syncthreads();                                         // end of the task
        if (warp == tileWarp) {
            if constexpr (MT == 0) {
                if (lane == 0) {
                    tma_reduce_add_4d(&tmPhi, smem_u32(sQ), 0, P.tm_rows * brick, 0, prob * P.Gs + P.g);
                    bulk_commit();
                }
            } else if (lane < NM) {
                float* gphi = P.phi + (size_t)(prob * P.Gs + P.g) * NM * P.cells_p + (size_t)brick * P.NCb;
                bulk_reduce_add_f32(gphi + (size_t)lane * P.cells_p, smem_u32(sQ + lane * NCP), uint32_t(NC * 4));
                bulk_commit();
            }
        }
        if (tid == 0 && (edge_x | edge_y | edge_z)) {
            float s = 0.0f;
            for (int w = 0; w < P.W; ++w) s += sRed[w];
            atomicAdd(P.leak + prob, (double)s);
        }
        if (publisher) {                                         // the other lanes of its warp are already on the next task
            bulk_wait0();                                        // the face blocks are in global memory
            fence_proxy_async_global();
            st_release_u32(flag_base + brick, P.epoch);
        }
    }
    if (warp == tileWarp) bulk_wait0();
}

}  // namespace doctors
