// a3-a5  Row-pipelined sweep kernel (sweep_mode 2): one persistent CTA per SM sweeps whole x-ROWS of bricks.
//
// Same two-level sub-sweep schedule as sweep_brick.cuh (Eq. 8 applied to the brick grid and to the
// cells of a brick), same arithmetic (dd_cell, FFMA2 projections, fp64 face recurrence), same global data (brick-major
// arrays, per-brick flags, y / z face buffers).  What changes is the shape of a task and the overlap inside a CTA:
//
//   task      = (problem, octant, bj, bk): the gbx bricks of one x-row, visited in sweep order.  The x face never
//               leaves the registers and the in-brick wavefront (lane (j',k') at step s -> cell i' = s - j' - k' of the
//               ROW) runs on across brick boundaries: fill / drain costs BY + BZ - 2 steps per row instead of per brick.
//   pipeline  = three tile buffers; while the 10 wavefront warps sweep brick c, projection warps run phase 0 of brick
//               c+1 and phase 2 of brick c-1, a loader lane keeps the tensor copies / reduce-adds two bricks ahead, two
//               poller lanes wait for the upwind rows (which run at least one brick ahead on other SMs) and fetch the
//               y / z inflow faces, a publisher lane stores the outflow faces and releases the brick's flag.
//               All of them walk the same "brick stream" (rows back to back), each at its own lag, synchronised by
//               mbarriers in shared memory; nothing in the stream ever waits for a downstream row, so it cannot deadlock.
//
// Restrictions (everything else runs through k_sweep_brick): M <= kMaxSweepWarps directions per octant, face blocks of a
// multiple of 16 bytes.
#pragma once
#include "sweep_brick.cuh"

namespace doctors {

constexpr int kRowRing = 8;           // brick descriptors of the stream kept in shared memory
constexpr int kRowTabRing = 4;        // octant table blobs kept in shared memory (a row names its slot)
// Two configurations (template parameters of the kernel):
//   A  one CTA per SM, 3 stages, 5 projection warps with 4 cells per thread (96 registers): no stage ever waited for
//   B  two CTAs per SM, 2 stages, 4 projection warps with 2 cells per thread (64 registers): twice the wavefront warps per
//      SM; a stage is recycled (phase 2 -> reduce-add -> next load -> phase 0) while the wavefront is on the other one
// The control warp's lanes 0..3 are the loader, the y poller, the z poller and the publisher.
template <int STAGES, int PW> constexpr int row_threads() { return 32 * (kMaxSweepWarps + PW + 1); }

struct RowParams {
    int nx, ny, nz;
    int BX, BY, BZ;
    int gbx, gby, gbz;
    int M;
    int nprob;
    int NCb;
    long long cells_p;
    int tm_rows;
    const double* sigt;              // [cells_p]
    const unsigned char* octtab;     // [8] blobs of octtab_layout(NM, M, 0)
    int g, Gs;
    unsigned epoch;
    int task_begin, ntasks;          // row tasks: x = prob | octant << 8, y = bj | bk << 10
    int counter_slot;
    const uint2* tasks;
    Control* ctl;
    unsigned* flags;                 // [prob][8][bricks]
    double* faceY;                   // [prob][8][gbx*gbz][M][BZ][BX]
    double* faceZ;                   // [prob][8][gbx*gby][M][BY][BX]
    const ProbState* state;
    double* leak;
    long long* dbg_time;             // -DDOCTORS_TIMING builds only: [16] cycle sums per role / wait
};

// One entry of the brick stream.
struct RowDesc {
    int prob, oct;
    int bi, bj, bk;                  // brick
    int first, last;                 // first / last brick of its row
    int stop;                        // 1: end of the stream (no brick)
    int tab;                         // slot of the octant's table blob in shared memory
    int pad[3];
};

struct RowSmem {
    size_t bars, desc, lead, tile, sig, face, tab, done, total;
};
__host__ __device__ inline RowSmem row_smem_layout(int NM, int BX, int BY, int BZ, int M, int stages)
{
    RowSmem s;
    const size_t NC = size_t(BX) * BY * BZ;
    size_t o = 0;
    s.bars = o;  o += 8 * 8 * size_t(stages);                    // 8 mbarrier kinds x stages
    s.desc = o;  o += sizeof(RowDesc) * kRowRing;
    s.lead = o;  o = align_up(o + 64, 128);
    s.tile = o;  o = align_up(o + stages * size_t(NM > M ? NM : M) * NC * 4, 128);
    s.sig = o;   o = align_up(o + stages * NC * 8, 128);
    s.face = o;  o = align_up(o + stages * size_t(M) * (size_t(BX) * BZ + size_t(BX) * BY) * 8, 128);
    s.tab = o;   o = align_up(o + kRowTabRing * octtab_layout(NM, M, 0).total, 16);
    s.done = o;  o = align_up(o + 256, 16);
    o = align_up(o + 128, 16);                                   // tail pad (idle lanes read past the end of their arrays)
    s.total = o;
    return s;
}

// mbarrier kinds (index = kind * STAGES + stage)
enum { kBarQ = 0,        // tile + sigma_t landed (tx bytes; armed by the loader)
       kBarPsi = 1,      // phase 0 done: q_n in place (projection warps arrive)
       kBarWave = 2,     // wavefront done on this tile: psi_n in place, outflow faces written (wavefront warps arrive)
       kBarPhi = 3,      // phase 2 done: phi contribution in place (projection warps arrive)
       kBarFace = 4,     // inflow faces landed (tx bytes; armed by the pollers, 2 arrivals)
       kBarFaceFree = 5, // publisher has read the outflow faces out of the slot
       kBarTileFree = 6, // loader: reduce-add has read the tile (loader arrives itself: keeps the phase logic uniform)
       kBarSpare = 7 };

__device__ __forceinline__ bool mbar_try(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ int lds_volatile_s32(uint32_t a)
{
    int v;
    asm volatile("ld.volatile.shared.s32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void sts_volatile_s32(uint32_t a, int v) { asm volatile("st.volatile.shared.s32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }


// ---- kernel ----------------------------------------------------------------------------------------------------
template <int NM, bool FIX, int STAGES, int PW, int CPT, int CTAS>
__global__ void __launch_bounds__((row_threads<STAGES, PW>()), CTAS)
k_sweep_row(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmPhi, const RowParams P)
{
    static_assert(NM <= 16, "moment planes");
    constexpr int kRowStages = STAGES, kRowProjWarps = PW;
    if (__ldcg(&P.ctl->all_done)) return;
    extern __shared__ __align__(128) unsigned char smem[];
    const int BX = P.BX, BY = P.BY, BZ = P.BZ, M = P.M;
    const int NC = BX * BY * BZ;
    const RowSmem L = row_smem_layout(NM, BX, BY, BZ, M, STAGES);
    const OctTab T = octtab_layout(NM, M, 0);
    const int planes = NM > M ? NM : M;
    const uint32_t sb = smem_u32(smem);
    const uint32_t tileBytes = uint32_t(planes) * NC * 4, sigBytes = uint32_t(NC) * 8;
    const int faceYn = M * BX * BZ, faceZn = M * BX * BY;          // doubles per brick
    const uint32_t faceBytes = uint32_t(faceYn + faceZn) * 8;
    auto bar_of = [&](int kind, int st) { return sb + uint32_t(L.bars) + 8u * uint32_t(kind * kRowStages + st); };
    auto tile_of = [&](int st) { return sb + uint32_t(L.tile) + uint32_t(st) * tileBytes; };
    auto sig_of = [&](int st) { return sb + uint32_t(L.sig) + uint32_t(st) * sigBytes; };
    auto facey_of = [&](int st) { return sb + uint32_t(L.face) + uint32_t(st) * faceBytes; };
    auto facez_of = [&](int st) { return sb + uint32_t(L.face) + uint32_t(st) * faceBytes + uint32_t(faceYn) * 8u; };
    RowDesc* sDesc = reinterpret_cast<RowDesc*>(smem + L.desc);
    const uint32_t leadAddr = sb + uint32_t(L.lead);
    unsigned char* sDoneP = smem + L.done;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int Wv = M;                                            // wavefront warps in use (one direction each)
    const int projW0 = kMaxSweepWarps, ctlW0 = kMaxSweepWarps + kRowProjWarps;
    const int nbricks = P.gbx * P.gby * P.gbz;

    if (tid == 0) {
        for (int st = 0; st < kRowStages; ++st) {
            mbar_init(bar_of(kBarQ, st), 1);
            mbar_init(bar_of(kBarPsi, st), kRowProjWarps);
            mbar_init(bar_of(kBarWave, st), Wv);
            mbar_init(bar_of(kBarPhi, st), kRowProjWarps);
            mbar_init(bar_of(kBarFace, st), 2);
            mbar_init(bar_of(kBarFaceFree, st), 1);
        }
        fence_mbar_init();
        sts_volatile_s32(leadAddr, 0);
    }
    // the stopped-problem bytes: once per launch
    for (int q = tid; q < P.nprob; q += blockDim.x) sDoneP[q] = (unsigned char)(__ldcg(&P.state[q].done) != 0);
    __syncthreads();

#ifdef DOCTORS_TIMING
    long long tw[4] = {0, 0, 0, 0};
    const long long tstart = clock64();
#define RT_BEGIN long long t0_ = clock64()
#define RT_END(i) tw[i] += clock64() - t0_
#define RT_FLUSH(base, who) do { if (who) { tw[0] = clock64() - tstart; for (int i_ = 0; i_ < 4; ++i_) atomicAdd(reinterpret_cast<unsigned long long*>(P.dbg_time) + (base) + i_, (unsigned long long)tw[i_]); } } while (0)
#else
#define RT_BEGIN do { } while (0)
#define RT_END(i) do { } while (0)
#define RT_FLUSH(base, who) do { } while (0)
#endif
    // wait until the loader has published stream position c, return its descriptor
    auto desc_at = [&](int c) -> RowDesc {
        while (lds_volatile_s32(leadAddr) <= c) { }
        __threadfence_block();
        return sDesc[c % kRowRing];
    };
    auto tab_of = [&](int slot) { return smem + L.tab + size_t(slot) * T.total; };

    // ================================================================================================================
    if (warp == ctlW0) {
        // ---- loader (lane 0): row tasks -> brick stream, tile loads ahead of phase 0, reduce-adds behind phase 2 ----
        if (lane == 0) {
            int tabslot = -1, taboct = -1;
            int c = 0;
            int next_id = int(atomicAdd(&P.ctl->counters[P.counter_slot], 1u));
            bool more = true;
            while (more) {
                // next row of a problem that still runs
                uint2 td = make_uint2(0u, 0u);
                bool have = false;
                while (next_id < P.ntasks) {
                    td = P.tasks[P.task_begin + next_id];
                    next_id = int(atomicAdd(&P.ctl->counters[P.counter_slot], 1u));
                    if (!sDoneP[td.x & 0xff]) { have = true; break; }
                }
                const int nb = have ? P.gbx : 1;                 // the stop marker takes one stream position
                const int oct = (td.x >> 8) & 7, sx = (oct & 1) ? -1 : 1;
                const bool newtab = have && oct != taboct;       // this row's octant tables are not in shared memory yet
                if (newtab) { taboct = oct; tabslot = (tabslot + 1) % kRowTabRing; }
                for (int i = 0; i < nb; ++i, ++c) {
                    RowDesc d;
                    d.prob = td.x & 0xff; d.oct = oct; d.bj = td.y & 0x3ff; d.bk = (td.y >> 10) & 0x3ff;
                    d.bi = sx > 0 ? i : P.gbx - 1 - i;
                    d.first = i == 0; d.last = i == nb - 1; d.stop = have ? 0 : 1; d.tab = tabslot;
                    sDesc[c % kRowRing] = d;
                    __threadfence_block();
                    sts_volatile_s32(leadAddr, c + 1);
                    const int st = c % kRowStages;
                    if (c >= kRowStages) {
                        // the tile of brick c-3 lives in this stage: wait for its phase 2, add it into phi, wait until read
                        const RowDesc o = sDesc[(c - kRowStages) % kRowRing];
                        { RT_BEGIN; mbar_wait(bar_of(kBarPhi, st), uint32_t((c - kRowStages) / kRowStages) & 1u); RT_END(1); }
                        const int ob = o.bi + P.gbx * (o.bj + P.gby * o.bk);
                        tma_reduce_add_4d(&tmPhi, tile_of(st), 0, P.tm_rows * ob, 0, o.prob * P.Gs + P.g);
                        bulk_commit();
                        { RT_BEGIN; bulk_wait_read0(); RT_END(2); }
                    }
                    if (have) {
                        const int brick = d.bi + P.gbx * (d.bj + P.gby * d.bk);
                        const bool tl = newtab && i == 0;          // the tables ride on the first brick's tile barrier
                        mbar_expect_tx(bar_of(kBarQ, st), uint32_t(NM * NC * 4 + NC * 8 + (tl ? T.total : 0)));
                        tma_load_4d(tile_of(st), &tmQ, bar_of(kBarQ, st), 0, P.tm_rows * brick, 0, d.prob);
                        bulk_load(sig_of(st), P.sigt + (size_t)brick * P.NCb, uint32_t(NC * 8), bar_of(kBarQ, st));
                        if (tl) bulk_load(smem_u32(tab_of(tabslot)), P.octtab + (size_t)oct * T.total, uint32_t(T.total), bar_of(kBarQ, st));
                    }
                }
                more = have;
            }
            // drain: the last bricks' reduce-adds (c is one past the stop marker)
            const int cend = c - 1;                              // position of the stop marker
            for (int o_ = (cend >= kRowStages ? cend - kRowStages + 1 : 0); o_ < cend; ++o_) {
                // bricks whose reduce has not been issued: those with o_ + kRowStages > cend  (the marker position itself handled o_ = cend - 3)
                if (o_ + kRowStages <= cend) continue;
                const int st = o_ % kRowStages;
                const RowDesc o = sDesc[o_ % kRowRing];
                mbar_wait(bar_of(kBarPhi, st), uint32_t(o_ / kRowStages) & 1u);
                const int ob = o.bi + P.gbx * (o.bj + P.gby * o.bk);
                tma_reduce_add_4d(&tmPhi, tile_of(st), 0, P.tm_rows * ob, 0, o.prob * P.Gs + P.g);
                bulk_commit();
            }
            bulk_wait0();
            RT_FLUSH(0, true);
        }
        else if (lane == 1 || lane == 2) {
            // ---- pollers (lane 1: y, lane 2: z): inflow faces of every brick of the stream ----
            const bool isz = lane == 2;
            for (int c = 0;; ++c) {
                const RowDesc d = desc_at(c);
                if (d.stop) break;
                const int st = c % kRowStages;
                if (c >= kRowStages) { RT_BEGIN; mbar_wait(bar_of(kBarFaceFree, st), uint32_t(c / kRowStages - 1) & 1u); RT_END(1); }
                const int sy = (d.oct & 2) ? -1 : 1, sz = (d.oct & 4) ? -1 : 1;
                const bool up = isz ? (sz > 0 ? d.bk > 0 : d.bk < P.gbz - 1) : (sy > 0 ? d.bj > 0 : d.bj < P.gby - 1);
                const uint32_t dst = isz ? facez_of(st) : facey_of(st);
                const int n8 = isz ? faceZn : faceYn;
                if (up) {
                    const int brick = d.bi + P.gbx * (d.bj + P.gby * d.bk);
                    const int upb = isz ? brick - sz * P.gbx * P.gby : brick - sy * P.gbx;
                    const size_t po = (size_t)d.prob * 8 + d.oct;
                    const unsigned* flag = P.flags + po * nbricks + upb;
                    const double* src = isz ? P.faceZ + (po * (P.gbx * P.gby) + d.bi + P.gbx * d.bj) * (size_t)faceZn
                                            : P.faceY + (po * (P.gbx * P.gbz) + d.bi + P.gbx * d.bk) * (size_t)faceYn;
                    { RT_BEGIN; while (ld_acquire_u32(flag) != P.epoch) { } RT_END(2); }
                    fence_proxy_async_all();
                    mbar_expect_tx(bar_of(kBarFace, st), uint32_t(n8) * 8u);
                    bulk_load(dst, src, uint32_t(n8) * 8u, bar_of(kBarFace, st));
                } else {
                    for (int e = 0; e < n8; ++e) sts_f64(dst + 8u * e, 0.0);   // vacuum
                    mbar_arrive(bar_of(kBarFace, st));
                }
            }
            RT_FLUSH(4, isz);
        }
        else if (lane == 3) {
            // ---- publisher (lane 3): outflow faces of every brick -> global, then the brick's flag ----
            {
            for (int c = 0;; ++c) {
                const RowDesc d = desc_at(c);
                if (d.stop) break;
                const int st = c % kRowStages;
                { RT_BEGIN; mbar_wait(bar_of(kBarWave, st), uint32_t(c / kRowStages) & 1u); RT_END(1); }
                const int sy = (d.oct & 2) ? -1 : 1, sz = (d.oct & 4) ? -1 : 1;
                const bool dny = sy > 0 ? d.bj < P.gby - 1 : d.bj > 0;
                const bool dnz = sz > 0 ? d.bk < P.gbz - 1 : d.bk > 0;
                const size_t po = (size_t)d.prob * 8 + d.oct;
                if (dny) bulk_store(P.faceY + (po * (P.gbx * P.gbz) + d.bi + P.gbx * d.bk) * (size_t)faceYn, facey_of(st), uint32_t(faceYn) * 8u);
                if (dnz) bulk_store(P.faceZ + (po * (P.gbx * P.gby) + d.bi + P.gbx * d.bj) * (size_t)faceZn, facez_of(st), uint32_t(faceZn) * 8u);
                bulk_commit();
                bulk_wait_read0();
                mbar_arrive(bar_of(kBarFaceFree, st));
                if (dny | dnz) {
                    { RT_BEGIN; bulk_wait0(); RT_END(2); }
                    fence_proxy_async_all();
                    st_release_u32(P.flags + po * nbricks + d.bi + P.gbx * (d.bj + P.gby * d.bk), P.epoch);
                }
            }
            }
            RT_FLUSH(8, true);
        }
    } else if (warp >= projW0 && warp < ctlW0) {
        // ---- projection warps: phase 0 of brick c+2, phase 2 of brick c (a5) ----
        const int pt = tid - 32 * projW0, pn = 32 * kRowProjWarps;
        auto phase0 = [&](int c, const RowDesc& d) {
            const int st = c % kRowStages;
            { RT_BEGIN; mbar_wait(bar_of(kBarQ, st), uint32_t(c / kRowStages) & 1u); RT_END(1); }
            float* sQ = reinterpret_cast<float*>(smem + L.tile + size_t(st) * tileBytes);
            const float* sM = reinterpret_cast<const float*>(tab_of(d.tab) + T.t0);
            for (int c0 = pt; c0 < NC; c0 += CPT * pn) {
                int cc[CPT]; bool ok[CPT];
#pragma unroll
                for (int u = 0; u < CPT; ++u) { cc[u] = c0 + u * pn; ok[u] = cc[u] < NC; }
                if constexpr (NM >= 2) {
                    float2 q[CPT][NM / 2];
                    float ql[CPT];
#pragma unroll
                    for (int u = 0; u < CPT; ++u) {
#pragma unroll
                        for (int k = 0; k < NM / 2; ++k)
                            q[u][k] = ok[u] ? make_float2(sQ[(2 * k) * NC + cc[u]], sQ[(2 * k + 1) * NC + cc[u]]) : make_float2(0.0f, 0.0f);
                        ql[u] = ((NM & 1) && ok[u]) ? sQ[(NM - 1) * NC + cc[u]] : 0.0f;
                    }
                    for (int n = 0; n < M; ++n) {
                        const float2* mt = reinterpret_cast<const float2*>(sM + n * kTabPitch<NM>());
                        float2 acc[CPT];
#pragma unroll
                        for (int u = 0; u < CPT; ++u) acc[u] = make_float2(0.0f, 0.0f);
#pragma unroll
                        for (int k = 0; k < NM / 2; ++k) {
                            const float2 m2 = mt[k];
#pragma unroll
                            for (int u = 0; u < CPT; ++u) acc[u] = __ffma2_rn(m2, q[u][k], acc[u]);
                        }
                        const float ml = (NM & 1) ? sM[n * kTabPitch<NM>() + NM - 1] : 0.0f;
#pragma unroll
                        for (int u = 0; u < CPT; ++u) {
                            float r = acc[u].x + acc[u].y;
                            if (NM & 1) r = fmaf(ml, ql[u], r);
                            if (ok[u]) sQ[n * NC + cc[u]] = r;       // in place: this thread has read all of its cells
                        }
                    }
                } else {
                    float q0[CPT];
#pragma unroll
                    for (int u = 0; u < CPT; ++u) q0[u] = ok[u] ? sQ[cc[u]] : 0.0f;
                    for (int n = 0; n < M; ++n) {
                        const float m0 = sM[n * kTabPitch<NM>()];
#pragma unroll
                        for (int u = 0; u < CPT; ++u) if (ok[u]) sQ[n * NC + cc[u]] = m0 * q0[u];
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_of(kBarPsi, st));
        };
        auto phase2 = [&](int c, const RowDesc& d) {
            const int st = c % kRowStages;
            { RT_BEGIN; mbar_wait(bar_of(kBarWave, st), uint32_t(c / kRowStages) & 1u); RT_END(2); }
            float* sQ = reinterpret_cast<float*>(smem + L.tile + size_t(st) * tileBytes);
            const float* sD = reinterpret_cast<const float*>(tab_of(d.tab) + T.t2);
            for (int c0 = pt; c0 < NC; c0 += CPT * pn) {
                int cc[CPT]; bool ok[CPT];
#pragma unroll
                for (int u = 0; u < CPT; ++u) { cc[u] = c0 + u * pn; ok[u] = cc[u] < NC; }
                if constexpr (NM >= 2) {
                    float2 pa[CPT][NM / 2];
                    float pl[CPT];
#pragma unroll
                    for (int u = 0; u < CPT; ++u) {
                        pl[u] = 0.0f;
#pragma unroll
                        for (int k = 0; k < NM / 2; ++k) pa[u][k] = make_float2(0.0f, 0.0f);
                    }
                    for (int n = 0; n < M; ++n) {
                        const float2* dt = reinterpret_cast<const float2*>(sD + n * kTabPitch<NM>());
                        float2 v2[CPT];
#pragma unroll
                        for (int u = 0; u < CPT; ++u) { const float v = ok[u] ? sQ[n * NC + cc[u]] : 0.0f; v2[u] = make_float2(v, v); }
#pragma unroll
                        for (int k = 0; k < NM / 2; ++k) {
                            const float2 d2 = dt[k];
#pragma unroll
                            for (int u = 0; u < CPT; ++u) pa[u][k] = __ffma2_rn(d2, v2[u], pa[u][k]);
                        }
                        if (NM & 1) {
                            const float dl = sD[n * kTabPitch<NM>() + NM - 1];
#pragma unroll
                            for (int u = 0; u < CPT; ++u) pl[u] = fmaf(dl, v2[u].x, pl[u]);
                        }
                    }
#pragma unroll
                    for (int u = 0; u < CPT; ++u) {
                        if (ok[u]) {
#pragma unroll
                            for (int k = 0; k < NM / 2; ++k) { sQ[(2 * k) * NC + cc[u]] = pa[u][k].x; sQ[(2 * k + 1) * NC + cc[u]] = pa[u][k].y; }
                            if (NM & 1) sQ[(NM - 1) * NC + cc[u]] = pl[u];
                        }
                    }
                } else {
                    float p0[CPT];
#pragma unroll
                    for (int u = 0; u < CPT; ++u) p0[u] = 0.0f;
                    for (int n = 0; n < M; ++n) {
                        const float d0 = sD[n * kTabPitch<NM>()];
#pragma unroll
                        for (int u = 0; u < CPT; ++u) if (ok[u]) p0[u] = fmaf(d0, sQ[n * NC + cc[u]], p0[u]);
                    }
#pragma unroll
                    for (int u = 0; u < CPT; ++u) if (ok[u]) sQ[cc[u]] = p0[u];
                }
            }
            fence_proxy_async_smem();                            // the reduce-add reads the tile through the async proxy
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_of(kBarPhi, st));
        };
        // order: P0(0), P0(1), then for c = 0, 1, ...: P2(c), P0(c + 2)
        bool ended = false;                                      // the stop marker has been seen by the P0 side
        for (int c = 0; c < 2 && !ended; ++c) {
            const RowDesc d = desc_at(c);
            if (d.stop) ended = true; else phase0(c, d);
        }
        for (int c = 0;; ++c) {
            const RowDesc d = desc_at(c);
            if (d.stop) break;
            phase2(c, d);
            if (!ended) {
                const RowDesc e = desc_at(c + 2);
                if (e.stop) ended = true; else phase0(c + 2, e);
            }
        }
        RT_FLUSH(12, tid == 32 * projW0);
    }
    else if (warp < Wv) {
        // ---- wavefront warps (a3 level 2, a4): warp = direction, lanes = (j',k'), step s -> cell x = s - j' - k' of the ROW ----
        const int n = warp;
        int jp, kp;
        lane_cross_section(lane, BY, jp, kp);
        const int skew = jp + kp;
        const int exLast = P.nx - (P.gbx - 1) * BX;              // cells of the clipped brick at the +x end of the row
        const int shy = BY;
        for (int c = 0;;) {
            const RowDesc d0 = desc_at(c);
            if (d0.stop) break;
            const int oct = d0.oct;
            const int sx = (oct & 1) ? -1 : 1, sy = (oct & 2) ? -1 : 1, sz = (oct & 4) ? -1 : 1;
            const int ey = min(BY, P.ny - d0.bj * BY), ez = min(BZ, P.nz - d0.bk * BZ);
            const bool lane_ok = kp < ez && jp < ey;
            const int lj = sy > 0 ? jp : ey - 1 - jp;
            const int lk_ = sz > 0 ? kp : ez - 1 - kp;
            const bool first_y = jp == 0, first_z = kp == 0, last_y = jp == ey - 1, last_z = kp == ez - 1;
            const bool edge_y = sy > 0 ? d0.bj == P.gby - 1 : d0.bj == 0;   // outflow faces on the mesh boundary
            const bool edge_z = sz > 0 ? d0.bk == P.gbz - 1 : d0.bk == 0;
            // the octant's tables ride on the tile barrier of the row's first brick (one phase ahead at most: safe to wait here)
            mbar_wait(bar_of(kBarQ, c % kRowStages), uint32_t(c / kRowStages) & 1u);
            const double* dir = reinterpret_cast<const double*>(tab_of(d0.tab) + T.dir) + 4 * n;
            const double cx = dir[0], cy = dir[1], cz = dir[2], cs = dir[3];
            const float4 lkc = reinterpret_cast<const float4*>(tab_of(d0.tab) + T.lk)[n];
            int nxr = P.nx, gbx = P.gbx;
            asm volatile("" : "+r"(nxr), "+r"(gbx));             // kept in registers: otherwise re-read from the constant bank every step
            auto len_of = [&](int i) { return (sx > 0 ? i : gbx - 1 - i) == gbx - 1 ? exLast : BX; };
            const int nsteps = nxr + ey + ez - 2;
            const int d4 = lane_ok ? 4 * sx : 0, d8 = 2 * d4;
            double ax = 0.0, oy = 0.0, oz = 0.0;                  // vacuum at the row's inflow x face
            double outy = 0.0, outz = 0.0;                       // sums of boundary outflow (leakage report)
            // lane state: its current brick of the row (visiting order), cells left in it, running addresses of its cell
            int cur = -1, rem = 0;
            uint32_t pq = tile_of(0) + 2048u, ps = pq, py = pq, pz = pq;
            int open_i = 0, open_at = 0;                         // lane (0,0) enters brick open_i at step open_at
            int close_i = 0, close_at = len_of(0) + ey + ez - 3; // after this step the last lane has left brick close_i
#pragma unroll 1
            for (int s = 0; s < nsteps; ++s) {
                if (s == open_at && open_i < gbx) {              // the brick's q_n and inflow faces must be there
                    const int pos = c + open_i, st = pos % kRowStages;
                    { RT_BEGIN; mbar_wait(bar_of(kBarPsi, st), uint32_t(pos / kRowStages) & 1u); RT_END(1); }
                    { RT_BEGIN; mbar_wait(bar_of(kBarFace, st), uint32_t(pos / kRowStages) & 1u); RT_END(2); }
                    open_at += len_of(open_i);
                    ++open_i;
                }
                const int xr = s - skew;                         // this lane's cell of the row, in sweep order
                const bool act = lane_ok && (unsigned)xr < (unsigned)nxr;
                if (act && rem == 0) {                           // this lane enters its next brick
                    ++cur;
                    const int ex_c = len_of(cur), st = (c + cur) % kRowStages;
                    rem = ex_c;
                    const int li0 = sx > 0 ? 0 : ex_c - 1;
                    const uint32_t rowoff = uint32_t(BX * (lj + BY * lk_) + li0);
                    pq = tile_of(st) + 4u * (uint32_t(n * NC) + rowoff);
                    ps = sig_of(st) + 8u * rowoff;
                    py = facey_of(st) + 8u * uint32_t((n * BZ + lk_) * BX + li0);
                    pz = facez_of(st) + 8u * uint32_t((n * BY + lj) * BX + li0);
                }
                double b = __shfl_up_sync(0xffffffffu, oy, 1);
                double cc = __shfl_up_sync(0xffffffffu, oz, shy);
                const float q = lds_f32(pq);
                const double sg = lds_f64(ps);
                if (first_y) b = lds_f64(py);
                if (first_z) cc = lds_f64(pz);
                double ox;
                const float psi = dd_cell<FIX>(act, q, sg, cx, cy, cz, cs, ax, b, cc, ox, oy, oz);
                sts_f32_if(act, pq, psi);
                sts_f64_if(act && last_y, py, oy);
                sts_f64_if(act && last_z, pz, oz);
                if (act) {
                    ax = ox; --rem;
                    if (edge_y && last_y) outy += oy;
                    if (edge_z && last_z) outz += oz;
                }
                pq += d4; ps += d8; py += d8; pz += d8;
                if (s == close_at) {                             // the last lane has left brick close_i
                    const int pos = c + close_i;
                    fence_proxy_async_smem();                    // outflow faces -> bulk store (async proxy)
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar_of(kBarWave, pos % kRowStages));
                    ++close_i;
                    close_at += close_i < gbx ? len_of(close_i) : (1 << 28);
                }
            }
            // leakage through the mesh boundary (balance report): w |Omega_d| A_d psi_out summed over boundary faces
            float lk = lane_ok ? lkc.x * (float)ax + lkc.y * (float)outy + lkc.z * (float)outz : 0.0f;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) lk += __shfl_xor_sync(0xffffffffu, lk, o);
            if (lane == 0) atomicAdd(P.leak + d0.prob, (double)lk);
            c += P.gbx;
        }
        RT_FLUSH(16, tid == 0);
    }
#undef RT_BEGIN
#undef RT_END
#undef RT_FLUSH
}

}  // namespace doctors
