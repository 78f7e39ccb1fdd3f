// Shared device-side types and small PTX wrappers (sm_100a).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdint>

namespace doctors {

constexpr int kMaxMaterials = 16;
constexpr int kMaxMoments = 16;       // P3
constexpr int kMaxSweepWarps = 10;   // sweep CTA = one warp per direction of the octant (looped if M > 10)

// Device storage order of every per-cell array is BRICK-MAJOR: cell (i,j,k) lives at
//   cp = brick * NCb + lj + BY*(li + BX*lk),  brick = bi + gbx*(bj + gby*bk),  (bi,li) = divmod(i, BX) ...
// so that the tile a sweep task loads (one brick, one moment) is ONE contiguous run of NCb*4 bytes
// instead of BY*BZ rows of BX*4 bytes (64-byte rows made the TMA unit fetch whole 128-byte lines: 2x
// read amplification on Q, measured in round 1).  INSIDE a brick y runs fastest, then x, then z: the
// wavefront's 32 lanes (j',k') touch, at step s, the cells i' = s - j' - k', i.e. local indices
// 8 s - 7 j' + 8 (BX - 1) k' for an 8 x 4 cross section — 32 different banks for every even BX (and 16
// different 8-byte bank pairs per half warp for sigma_t).  With x fastest the same lanes sat at
// (BX - 1) j' + (BX BY - 1) k', which collides for every even BX: 21 % of the shared-memory wavefronts of the
// round-1 kernel were bank-conflict replays (profiles/r02_sweep_ncu.md).
// Bricks at the mesh edge are padded with inert cells (density 0, all fields 0).  The ray tracer alone also
// reads dense x-fastest copies of material / density.
struct MeshDev {
    int nx, ny, nz;
    int BX, BY, BZ;         // brick extents
    int gbx, gby, gbz;      // brick grid
    int NCb;                // cells per brick
    long long cells_p;      // gbx*gby*gbz*NCb (padded cell count)
    double dx, dy, dz;
    double x0, y0, z0;      // centre of cell (0,0,0)
};
__host__ __device__ __forceinline__ long long cell_index(const MeshDev& m, int i, int j, int k)
{
    const int bi = i / m.BX, bj = j / m.BY, bk = k / m.BZ;
    const int li = i - bi * m.BX, lj = j - bj * m.BY, lk = k - bk * m.BZ;
    return (long long)(bi + m.gbx * (bj + m.gby * bk)) * m.NCb + lj + m.BY * (li + m.BX * lk);
}
// returns false for a padding cell
__host__ __device__ __forceinline__ bool cell_ijk(const MeshDev& m, long long cp, int& i, int& j, int& k)
{
    const int brick = int(cp / m.NCb), local = int(cp - (long long)brick * m.NCb);
    const int lj = local % m.BY, t = local / m.BY, li = t % m.BX, lk = t / m.BX;
    const int bi = brick % m.gbx, u = brick / m.gbx, bj = u % m.gby, bk = u / m.gby;
    i = bi * m.BX + li; j = bj * m.BY + lj; k = bk * m.BZ + lk;
    return i < m.nx && j < m.ny && k < m.nz;
}

struct SourceDev {
    int kind;               // 0 volume, 1 point, 2 cone, 3 fan
    int vol_slot;           // kind 0: index into the volume-source array, else -1
    double pos[3];
    double axis[3];         // normalised
    double cos_half;
    double fan_n[3];        // kind 3: unit normal of the fan plane (perpendicular to axis)
    double sin_half2;       // kind 3: sine of the polar half angle
};

// Per-problem iteration state, device resident (row a6).
struct ProbState {
    unsigned max_diff_bits; // max |phi0_new - phi0_old| as float bits (non-negative floats order like uints)
    unsigned max_phi_bits;  // max |phi0_new|
    int iters;              // sweeps done for the current group
    int done;               // 1: this problem's current group has stopped
    int fixed;              // > 0: stop exactly at this sweep count
    int hit_max;            // stopped by max_iters
    float resid;            // last delta_k
    int pad;
};

struct Control {
    unsigned ticket;        // last-block election of k_check
    int all_done;           // every problem of the chunk is done for the current group
    unsigned counters[10];  // task counters of the sweep launches of one iteration
    unsigned pad[4];
};

// ---- small PTX wrappers ------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p)
{
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// named block barrier 1, split: bar_arrive1 does not wait (the publishing warp), bar_sync1 does
__device__ __forceinline__ void bar_sync1(int nthreads) { asm volatile("bar.sync 1, %0;" ::"r"(nthreads) : "memory"); }
__device__ __forceinline__ void bar_arrive1(int nthreads) { asm volatile("bar.arrive 1, %0;" ::"r"(nthreads) : "memory"); }
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok = 0;
    while (!ok) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok)
            : "r"(bar), "r"(parity)
            : "memory");
    }
}
__device__ __forceinline__ void fence_proxy_async_smem()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void tma_load_5d(uint32_t dst, const CUtensorMap* map, uint32_t bar,
                                            int c0, int c1, int c2, int c3, int c4)
{
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes"
        " [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
        ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(bar),
          "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
        : "memory");
}
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2, int c3)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes"
        " [%0], [%1, {%3, %4, %5, %6}], [%2];"
        ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
        : "memory");
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes"
        " [%0], [%1, {%3, %4}], [%2];"
        ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(bar), "r"(c0), "r"(c1)
        : "memory");
}
__device__ __forceinline__ void tma_reduce_add_4d(const CUtensorMap* map, uint32_t src, int c0, int c1, int c2, int c3)
{
    asm volatile(
        "cp.reduce.async.bulk.tensor.4d.global.shared::cta.add.tile.bulk_group"
        " [%0, {%2, %3, %4, %5}], [%1];"
        ::"l"(reinterpret_cast<uint64_t>(map)), "r"(src), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
        : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, uint32_t bar,
                                            int c0, int c1, int c2)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes"
        " [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(bar), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
}
// smem tile += into global through the TMA unit (L2 does the fp32 adds)
__device__ __forceinline__ void tma_reduce_add_5d(const CUtensorMap* map, uint32_t src,
                                                  int c0, int c1, int c2, int c3, int c4)
{
    asm volatile(
        "cp.reduce.async.bulk.tensor.5d.global.shared::cta.add.tile.bulk_group"
        " [%0, {%2, %3, %4, %5, %6}], [%1];"
        ::"l"(reinterpret_cast<uint64_t>(map)), "r"(src),
          "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
        : "memory");
}
__device__ __forceinline__ void tma_store_5d(const CUtensorMap* map, uint32_t src,
                                             int c0, int c1, int c2, int c3, int c4)
{
    asm volatile(
        "cp.async.bulk.tensor.5d.global.shared::cta.tile.bulk_group"
        " [%0, {%2, %3, %4, %5, %6}], [%1];"
        ::"l"(reinterpret_cast<uint64_t>(map)), "r"(src),
          "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
        : "memory");
}
__device__ __forceinline__ void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }
// generic <-> async proxy ordering for GLOBAL memory only (flags vs bulk copies of the face buffers)
__device__ __forceinline__ void fence_proxy_async_global() { asm volatile("fence.proxy.async.global;" ::: "memory"); }
// 1-D bulk copies through the TMA unit (no tensor map): size and both addresses multiples of 16 bytes
__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void bulk_store(void* dst, uint32_t src, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(bytes) : "memory");
}
// shared -> global elementwise fp32 add through the TMA unit (the adds happen in L2)
__device__ __forceinline__ void bulk_reduce_add_f32(float* dst, uint32_t src, uint32_t bytes)
{
    asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f32 [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

__device__ __forceinline__ float lds_f32(uint32_t a)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ double lds_f64(uint32_t a)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void sts_f32(uint32_t a, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory"); }
__device__ __forceinline__ void sts_f64(uint32_t a, double v) { asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v) : "memory"); }

__device__ __forceinline__ void sts_f32_if(bool p, uint32_t a, float v)
{
    asm volatile("{\n\t.reg .pred pp;\n\tsetp.ne.b32 pp, %0, 0;\n\t@pp st.shared.f32 [%1], %2;\n\t}" ::"r"((int)p), "r"(a), "f"(v) : "memory");
}
__device__ __forceinline__ void sts_f64_if(bool p, uint32_t a, double v)
{
    asm volatile("{\n\t.reg .pred pp;\n\tsetp.ne.b32 pp, %0, 0;\n\t@pp st.shared.f64 [%1], %2;\n\t}" ::"r"((int)p), "r"(a), "d"(v) : "memory");
}

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_u32(unsigned* p, unsigned v)
{
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// ---- tensor-core helpers for the 16-wide projections (legacy warp-level mma, TF32 operands, fp32 accumulate) ----
// D(16x8) += A(16x8, row) * B(8x8, col).  Fragment ownership (g = lane >> 2, t = lane & 3):
//   a0 (g, t)  a1 (g+8, t)  a2 (g, t+4)  a3 (g+8, t+4);   b0 (k = t, n = g)  b1 (k = t+4, n = g);
//   d0 (g, 2t)  d1 (g, 2t+1)  d2 (g+8, 2t)  d3 (g+8, 2t+1).
__device__ __forceinline__ void mma_tf32(float (&d)[4], const float4& a, float b0, float b1)
{
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
                 : "r"(__float_as_uint(a.x)), "r"(__float_as_uint(a.y)), "r"(__float_as_uint(a.z)), "r"(__float_as_uint(a.w)),
                   "r"(__float_as_uint(b0)), "r"(__float_as_uint(b1)));
}
// v = hi + lo with hi exactly representable in TF32 (rounded to nearest: add half an ulp, clear 13 bits — plain
// integer ALU; cvt.rna.tf32.f32 expands to four instructions here); lo = v - hi is exact in fp32, of either
// sign, and is truncated to TF32 by the tensor core: |v - hi - tf32(lo)| <= 2^-21 |v|, unbiased
__device__ __forceinline__ void split_tf32(float v, float& hi, float& lo)
{
    hi = __uint_as_float((__float_as_uint(v) + 0x1000u) & 0xffffe000u);
    lo = v - hi;
}
__device__ __forceinline__ float4 lds_v4f32(uint32_t a)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a) : "memory");
    return v;
}
// 3-product split: acc += a * b with a = (ah, al), b = (bh, bl); small terms first
__device__ __forceinline__ void mma_3xtf32(float (&d)[4], const float4& ah, const float4& al, float bh0, float bh1, float bl0, float bl1)
{
    mma_tf32(d, al, bh0, bh1);
    mma_tf32(d, ah, bl0, bl1);
    mma_tf32(d, ah, bh0, bh1);
}
__device__ __forceinline__ void sts_v2f32(uint32_t a, float x, float y) { asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(a), "f"(x), "f"(y) : "memory"); }

// ---- one cell, one direction: diamond difference (readings R1, R2) -----------
//   psi = (q + cx a + cy b + cz c) / (sigt + cx + cy + cz),  out_d = 2 psi - in_d
// FIX: any negative outflow is set to zero and the cell balance re-solved with that face's
// diamond relation dropped (its inflow then enters with weight c_d / 2); repeat while a new
// face flips.  Conserves the cell balance exactly.
//
// Precision: the face recurrence runs in fp64.  out_d = 2 psi - in_d cancels
// wherever sigma_t Delta / (2|Omega_d|) is near 1, so fp32 faces, fp32-rounded c_d or sigma_t
// perturb deep, strongly attenuated cells by up to 2e-4 (measured on config 4, groups 45-46);
// with fp64 faces, exact c_d and sigma_t = (double)rho * sigt_hat the same cells agree to 1e-5.
// The source q_n, the cell flux psi handed to the moment sums and all stored moments stay fp32.
__device__ __forceinline__ double rcp_f64(double d)
{
    // MUFU.RCP64H seed (measured on B200: relative error 2^-20.0) + one Newton step in fp64: 2^-39.9 = 9.7e-13 measured.
    // A cubic step (2^-60) costs one more DFMA on the critical chain of every cell and changes no parity figure
    // (config 4, groups 45-46: 9.9e-6 either way): the recurrence amplifies errors of 1e-12 to ~1e-8 at most.
    double r0;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r0) : "d"(d));
    const double e = fma(-d, r0, 1.0);
    return fma(r0, e, r0);
}

// Fix-up (reading R2): a face whose outflow went negative is set to zero and its diamond relation dropped — its inflow
// then enters the balance with weight c_d / 2 instead of c_d and c_d leaves the denominator; repeated while a new face
// flips (at most 3 solves: there are 3 faces).  Conserves the cell balance exactly.
// The face flags act through multipliers (h_d = 1/2 or 1 on the inflow term, m_d = 0 or 1 on c_d and on the outflow)
// built from one 32-bit select each: selects on fp64 values cost two instructions per value and made this path 62
// instructions per pass, which 23 % of the wavefront steps of config 4 execute.
__device__ __forceinline__ double dd_fixup(double dq, double sig, double cx, double cy, double cz,
                                           double ta, double tb, double tc, double a, double b, double c,
                                           double& ox, double& oy, double& oz)
{
    // flags as integer masks (all ones = flagged) taken from the sign bits: the compiler keeps these off the fp64 pipe
    int fx = __double2hiint(ox) >> 31, fy = __double2hiint(oy) >> 31, fz = __double2hiint(oz) >> 31;
    double psi = 0.0;
#pragma unroll 1
    for (int pass = 0; pass < 3; ++pass) {
        // h = 1/2 (0x3fe00000) if flagged else 1 (0x3ff00000);  m = 0 if flagged else 1
        const double hx = __hiloint2double(fx * 0x100000 + 0x3ff00000, 0), mx = __hiloint2double(0x3ff00000 & ~fx, 0);
        const double hy = __hiloint2double(fy * 0x100000 + 0x3ff00000, 0), my = __hiloint2double(0x3ff00000 & ~fy, 0);
        const double hz = __hiloint2double(fz * 0x100000 + 0x3ff00000, 0), mz = __hiloint2double(0x3ff00000 & ~fz, 0);
        const double n2 = fma(hz, tc, fma(hy, tb, fma(hx, ta, dq)));
        const double d2 = fma(mz, cz, fma(my, cy, fma(mx, cx, sig)));
        psi = n2 * rcp_f64(d2);
        ox = mx * fma(2.0, psi, -a);
        oy = my * fma(2.0, psi, -b);
        oz = mz * fma(2.0, psi, -c);
        // newly negative faces (a flagged face gives +-0: masked out)
        const int nx_ = (__double2hiint(ox) >> 31) & ~fx, ny_ = (__double2hiint(oy) >> 31) & ~fy, nz_ = (__double2hiint(oz) >> 31) & ~fz;
        if ((nx_ | ny_ | nz_) == 0) break;
        fx |= nx_; fy |= ny_; fz |= nz_;
    }
    return psi;
}

// `act` = this lane holds a real cell; idle lanes of the warp-wavefront compute on stale values and
// must not trigger fix-up passes.
template <bool FIX>
__device__ __forceinline__ float dd_cell(bool act, float q, double sig, double cx, double cy, double cz, double csum,
                                         double a, double b, double c, double& ox, double& oy, double& oz)
{
    // numerator as an FMA chain (the late arrivals b, c enter last: two dependent FMAs instead of multiply + two adds)
    const double dq = (double)q;
    double psi = fma(cz, c, fma(cy, b, fma(cx, a, dq))) * rcp_f64(sig + csum);
    ox = fma(2.0, psi, -a);
    oy = fma(2.0, psi, -b);
    oz = fma(2.0, psi, -c);
    if (FIX) {
        // any negative outflow?  (sign bits; -0.0 takes the slow path too, which then changes nothing)
        const int sgn = __double2hiint(ox) | __double2hiint(oy) | __double2hiint(oz);
        if (act && sgn < 0) psi = dd_fixup(dq, sig, cx, cy, cz, cx * a, cy * b, cz * c, a, b, c, ox, oy, oz);
    }
    return (float)psi;
}

}  // namespace doctors
