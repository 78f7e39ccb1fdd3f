// C ABI of the B200-native DOCTORS hot path (include/doctors_b200.h): host state machine,
// workspace planning, launch sequencing.  Every arithmetic step of the path runs in the
// kernels of kernels.cuh / sweep_brick.cuh; this file only validates, lays out memory and
// enqueues work on the caller's stream.
#include "../../include/doctors_b200.h"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include <nvtx3/nvToolsExt.h>

#include "device_common.cuh"
#include "host_tables.h"
#include "kernels.cuh"
#include "sweep_brick.cuh"

using namespace doctors;

namespace {

struct SourceHost {
    int kind = 0;
    double pos[3] = {0, 0, 0}, axis[3] = {1, 0, 0}, half = 0;
    double fan_n[3] = {0, 0, 1}, half2 = 0;
    std::vector<double> spectrum;
    std::vector<float> volume;
};

struct GroupResult { int iters; int hit_max; float resid; float pad; double leak; double bal_src; double bal_col; };

// Workspace layout for one choice of options.
struct Plan {
    bool ok = false;
    long long cells_p = 0; int NCb = 0; int tm_inner = 0, tm_rows = 0;   // TMA box = tm_rows rows of tm_inner cells = one brick
    int MT = 0;                     // m-tiles of the tensor-core projections (0: FFMA2 loops), see sweep_brick.cuh
    unsigned fbytes = 8;            // bytes per exchanged face value: 4 with closure 1, 8 with closure 0 (sweep_brick.cuh, FaceOf)
    int nprob = 0, chunk = 0, nchunks = 0, nsrc = 0, nvol = 0;
    int G = 0, L = 0, NM = 0, ndir = 0, M = 0;
    int mode = 0, sweep_mode = 0, deterministic = 0;
    int B[3] = {0, 0, 0}, gb[3] = {0, 0, 0};
    int W = 1;                      // sweep warps per CTA
    long long nbricks = 0, ntasks = 0;
    size_t smem = 0;
    // offsets
    size_t o_mat, o_rho, o_sigt_hat, o_sigs, o_spec, o_srcs, o_extvol, o_mtab, o_dtab, o_lk,
        o_sigt, o_Q, o_fixed, o_phi0old, o_phiall, o_phi0all, o_phiu, o_state, o_ctl, o_leak, o_bal,
        o_matd, o_rhod, o_scratch, o_results, o_fixediters, o_tasks, o_flags, o_fx, o_fy, o_fz, o_dird, o_dbg, o_sched, o_ox, o_oy, o_oz, o_octtab, o_resp;
    size_t face_x_n = 0, face_y_n = 0, face_z_n = 0;
    size_t total = 0;
};

struct SweepLaunch {
    CUtensorMap tmQ, tmPhi;
    BrickParams bp;
    int grid = 0;
    size_t smem = 0;
};

// What the device-side set-up (bricked mesh, tables, task list, tensor maps) was built for: a solve re-uses it when
// nothing of this changed since, so a second solve on unchanged inputs uploads only the fixed sweep counts.
struct PrepKey {
    unsigned long long inputs_version = 0;
    void* ws = nullptr;
    size_t total = 0;
    int chunk = 0, B[3] = {0, 0, 0}, MT = 0, sweep_mode = 0, deterministic = 0, closure = 0, ctas_opt = 0;
    bool operator==(const PrepKey& k) const
    {
        return inputs_version == k.inputs_version && ws == k.ws && total == k.total && chunk == k.chunk && B[0] == k.B[0] &&
               B[1] == k.B[1] && B[2] == k.B[2] && MT == k.MT && sweep_mode == k.sweep_mode && deterministic == k.deterministic &&
               closure == k.closure && ctas_opt == k.ctas_opt;
    }
};

}  // namespace

struct doctors_problem {
    int device = 0;
    cudaStream_t stream = nullptr;
    int num_sms = 0;
    std::string err;
    // inputs (copied)
    bool has_mesh = false, has_xs = false, has_quad = false, has_src = false;
    int nx = 0, ny = 0, nz = 0, n_mat_mesh = 0;
    double dx = 0, dy = 0, dz = 0;
    std::vector<uint8_t> mat;
    std::vector<float> rho;
    int n_mat_xs = 0, G = 0, L = 0;
    std::vector<double> sigt, sigs;
    int ndir = 0;
    std::vector<double> omega, w;
    int mode = 0;
    std::vector<SourceHost> sources;
    // workspace
    void* ws = nullptr;
    size_t ws_bytes = 0;
    unsigned long long inputs_version = 1;   // bumped by every set_* call
    // device-side set-up, cached between solves (prepare())
    bool prepared = false;
    PrepKey prep_key;
    MeshDev md;                              // with pitch and origin (the ray tracer, the fixed source)
    SweepLaunch SL;
    std::vector<int> oct_begin;              // slices of the task list (one per launch of an iteration)
    std::vector<std::vector<int32_t>> sched_off;   // sweep_mode 1: plane offsets per octant
    int ctas_per_sm = 0;
    unsigned epoch = 0;                      // "brick done" value of the last sweep launch; grows across solves
    int pl_inexact = 0;                      // the quadrature does not integrate Y_lm Y_l'm' exactly up to the P_L order set
    std::vector<cudaEvent_t> ev_pool;        // timing events, owned by the handle (no leak on an error return)
    size_t ev_used = 0;
    int* h_flag = nullptr;                   // pinned word for the convergence flag
    // result bookkeeping
    bool solved = false;
    Plan plan;
    MeshDev mesh_dev;
    int last_chunk_first = 0, last_chunk_count = 0;
    CUresult (*encode)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                       const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                       CUtensorMapL2promotion, CUtensorMapFloatOOBfill) = nullptr;
};

namespace {

// NVTX range around a phase of doctors_solve (host side; shows up in nsys / ncu timelines, costs nothing without a tool)
struct NvtxRange {
    explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
    NvtxRange(const NvtxRange&) = delete;
    NvtxRange& operator=(const NvtxRange&) = delete;
};

int fail(doctors_problem* p, int code, const char* fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (p) p->err = buf;
    return code;
}

#define CK(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(p, DOCTORS_CUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)

int nprob_of(const doctors_problem* p) { return p->mode == 0 ? int(p->sources.size()) : 1; }

// max | sum_n w_n Y_lm (2l'+1)/(4 pi) Y_l'm' - delta | over all moment pairs up to P_L (Galerkin identity D^T M = I)
double galerkin_defect(int L, const std::vector<double>& omega, const std::vector<double>& w)
{
    std::vector<double> Mt, Dt;
    projection_tables(L, omega, w, Mt, Dt);
    const int NM = (L + 1) * (L + 1), nd = int(w.size());
    double worst = 0.0;
    for (int a = 0; a < NM; ++a)
        for (int b = 0; b < NM; ++b) {
            double acc = 0.0;
            for (int n = 0; n < nd; ++n) acc += Dt[size_t(n) * NM + a] * Mt[size_t(n) * NM + b];
            worst = std::max(worst, std::fabs(acc - (a == b ? 1.0 : 0.0)));
        }
    return worst;
}
constexpr double kGalerkinTol = 1e-9;

// projection = 2: tensor cores where they apply; 0 (automatic): tensor cores for more than 16 directions per octant
// (S12, S16: measured on config 3, S16 P3, 619.6 against 730.3 ms per solve), the FMA loops below (config 4, S8: 4-7 %
// faster than the tensor-core path); 1: always the FMA loops.
bool wants_mma(const doctors_solve_opts* o, int M)
{
    const int pr = o ? o->projection : 0;
    return pr == 2 || (pr == 0 && M > 16);
}

void auto_brick(int NM, int M, int nx, int ny, int nz, const int* req, bool mt, unsigned fbytes, int B[3])
{
    if (req && req[0] > 0 && req[1] > 0 && req[2] > 0) { B[0] = req[0]; B[1] = req[1]; B[2] = req[2]; return; }
    // cross section = the 32 lanes of a warp (8 x 4, reshaped for thin meshes); BX as long as shared memory allows
    B[1] = std::min(8, ny);
    B[2] = std::min(32 / B[1], nz);
    if (B[2] < 4 && B[1] < ny) B[1] = std::min(32 / B[2], ny);
    const int cand[5] = {20, 16, 12, 8, 4};        // 20 x 8 x 4 = 640 cells = 2 per thread of a 320-thread CTA, 3 CTAs per SM
                                                    // (24 x 8 x 4 also fits three CTAs with fp32 exchange faces: measured equal, 8.61 ms)
    auto fits = [&](int bx, size_t limit) {
        return brick_smem_layout(NM, bx, B[1], B[2], M, mt ? projection_mtiles(NM, M, bx * B[1] * B[2]) : 0, fbytes).total <= limit;
    };
    for (int c = 0; c < 5; ++c) {
        B[0] = std::min(cand[c], (nx + 3) / 4 * 4);
        if (fits(B[0], 74 * 1024)) break;
    }
    // many directions per octant (S16: 36 planes per tile): a brick shorter than 8 cells leaves 70 % of the wavefront's
    // lane-steps idle; two CTAs per SM with 8-cell bricks are faster (config 3: 2.86 against 3.47 ms per sweep)
    if (B[0] < 8 && nx > 4)
        for (int c = 0; c < 5; ++c) {
            const int bx = std::min(cand[c], (nx + 3) / 4 * 4);
            if (fits(bx, 113 * 1024)) { B[0] = bx; break; }
        }
}

// Lay out the workspace.  chunk = problems solved together.
Plan make_plan(const doctors_problem* p, const doctors_solve_opts* o, int chunk)
{
    Plan P;
    P.nprob = nprob_of(p);
    P.nsrc = int(p->sources.size());
    P.chunk = std::max(1, std::min(chunk, P.nprob));
    P.nchunks = (P.nprob + P.chunk - 1) / P.chunk;
    P.G = p->G; P.L = p->L; P.NM = (p->L + 1) * (p->L + 1);
    P.ndir = p->ndir; P.M = p->ndir / 8;
    P.mode = p->mode;
    P.sweep_mode = o ? o->sweep_mode : 0;
    P.deterministic = o ? o->deterministic : 0;
    for (auto& s : p->sources) if (s.kind == 0) ++P.nvol;
    P.fbytes = face_bytes(o && o->closure == 1);
    auto_brick(P.NM, P.M, p->nx, p->ny, p->nz, o ? o->brick : nullptr, wants_mma(o, P.M), P.fbytes, P.B);
    P.gb[0] = (p->nx + P.B[0] - 1) / P.B[0];
    P.gb[1] = (p->ny + P.B[1] - 1) / P.B[1];
    P.gb[2] = (p->nz + P.B[2] - 1) / P.B[2];
    P.nbricks = (long long)P.gb[0] * P.gb[1] * P.gb[2];
    P.NCb = P.B[0] * P.B[1] * P.B[2];
    P.cells_p = P.nbricks * P.NCb;                              // brick-major storage, edge bricks padded
    // one brick = NCb contiguous cells per moment; a TMA box row holds at most 256 elements and must be a 16-byte multiple
    P.tm_rows = 1;
    while ((P.NCb / 4) % P.tm_rows != 0 || P.NCb / P.tm_rows > 256) ++P.tm_rows;
    P.tm_inner = P.NCb / P.tm_rows;
    P.ntasks = P.nbricks * 8 * P.chunk;
    P.MT = wants_mma(o, P.M) ? projection_mtiles(P.NM, P.M, P.NCb) : 0;
    P.smem = brick_smem_layout(P.NM, P.B[0], P.B[1], P.B[2], P.M, P.MT, P.fbytes).total;
    { int dpw = (P.M + kMaxSweepWarps - 1) / kMaxSweepWarps; P.W = (P.M + dpw - 1) / dpw; }

    size_t off = 0;
    auto take = [&](size_t bytes) { size_t r = off; off = align_up(off + bytes, 256); return r; };
    const size_t cp = size_t(P.cells_p), nm = size_t(P.NM), G = size_t(P.G);
    // the memory in a mode-1 chunk: sources of the chunk = all sources
    const size_t src_per_chunk = P.mode == 0 ? size_t(P.chunk) : size_t(P.nsrc);
    (void)src_per_chunk;
    P.o_mat = take(cp);
    P.o_rho = take(cp * 4);
    P.o_matd = take(size_t(p->nx) * p->ny * p->nz);              // dense copies for the ray tracer
    P.o_rhod = take(size_t(p->nx) * p->ny * p->nz * 4);
    P.o_scratch = take(size_t(p->nx) * p->ny * p->nz * 4 * nm);  // get_*: dense staging of one (problem, group)
    P.o_sigt_hat = take(size_t(p->n_mat_xs) * G * 8);
    P.o_sigs = take(size_t(p->n_mat_xs) * (P.L + 1) * G * G * 4);
    P.o_spec = take(size_t(P.nsrc) * G * 8);
    P.o_srcs = take(size_t(P.nsrc) * sizeof(SourceDev));
    P.o_extvol = take(size_t(P.nvol) * G * cp * 4);
    P.o_mtab = take(size_t(P.ndir) * nm * 4);
    P.o_dtab = take(size_t(P.ndir) * nm * 4);
    P.o_lk = take(size_t(P.ndir) * 16);
    P.o_dird = take(size_t(P.ndir) * 32);
    P.o_sigt = take(cp * 8);
    P.o_Q = take(size_t(P.chunk) * nm * cp * 4);
    P.o_fixed = take(size_t(P.chunk) * nm * cp * 4);
    P.o_phi0old = take(size_t(P.chunk) * cp * 4);
    P.o_phiall = take(size_t(P.chunk) * G * nm * cp * 4);
    P.o_phi0all = take(size_t(P.nprob) * G * cp * 4);
    P.o_phiu = take(size_t(P.nsrc) * G * cp * 4);
    P.o_state = take(size_t(P.chunk) * sizeof(ProbState));
    P.o_ctl = take(sizeof(Control));
    P.o_leak = take(size_t(P.chunk) * 8);
    P.o_bal = take(size_t(P.chunk) * 16);
    P.o_results = take(size_t(P.nprob) * G * sizeof(GroupResult));
    P.o_fixediters = take(size_t(P.nprob) * G * 4);
    P.o_resp = take(G * 8);
    if (P.sweep_mode == 0) {
        P.face_x_n = size_t(P.M) * P.B[1] * P.B[2];
        P.face_y_n = size_t(P.M) * P.B[0] * P.B[2];
        P.face_z_n = size_t(P.M) * P.B[0] * P.B[1];
        P.o_tasks = take(size_t(P.ntasks) * sizeof(uint2));
        P.o_flags = take(size_t(P.chunk) * 8 * P.nbricks * 4);
        P.o_fx = take(size_t(P.chunk) * 8 * P.gb[1] * P.gb[2] * P.face_x_n * P.fbytes);
        P.o_fy = take(size_t(P.chunk) * 8 * P.gb[0] * P.gb[2] * P.face_y_n * P.fbytes);
        P.o_fz = take(size_t(P.chunk) * 8 * P.gb[0] * P.gb[1] * P.face_z_n * P.fbytes);
        P.o_dbg = take(size_t(P.B[0]) * P.B[1] * P.B[2] * 4);
        P.o_octtab = take(8 * octtab_layout(P.NM, P.M, P.MT).total);
        P.o_sched = P.o_ox = P.o_oy = P.o_oz = 0;
    } else {
        P.o_sched = take(size_t(8) * p->nx * p->ny * p->nz * 4);
        P.o_ox = take(size_t(P.chunk) * P.M * cp * 8);
        P.o_oy = take(size_t(P.chunk) * P.M * cp * 8);
        P.o_oz = take(size_t(P.chunk) * P.M * cp * 8);
        P.o_tasks = P.o_flags = P.o_fx = P.o_fy = P.o_fz = P.o_dbg = P.o_octtab = 0;
    }
    P.total = off;
    P.ok = true;
    return P;
}

int check_ready(doctors_problem* p)
{
    if (!p->has_mesh) return fail(p, DOCTORS_BAD_STATE, "mesh/materials not set");
    if (!p->has_xs) return fail(p, DOCTORS_BAD_STATE, "cross sections not set");
    if (!p->has_quad) return fail(p, DOCTORS_BAD_STATE, "quadrature not set");
    if (!p->has_src) return fail(p, DOCTORS_BAD_STATE, "source not set");
    if (p->n_mat_mesh > p->n_mat_xs)
        return fail(p, DOCTORS_BAD_STATE, "mesh uses %d materials, XS table has %d", p->n_mat_mesh, p->n_mat_xs);
    for (size_t s = 0; s < p->sources.size(); ++s) {
        const SourceHost& S = p->sources[s];
        if (S.kind == 0) {
            if (S.volume.size() != size_t(p->G) * p->nx * p->ny * p->nz)
                return fail(p, DOCTORS_BAD_STATE, "source %zu: volume array does not match G x mesh", s);
        } else if (S.spectrum.size() != size_t(p->G)) {
            return fail(p, DOCTORS_BAD_STATE, "source %zu: spectrum length %zu != G = %d", s, S.spectrum.size(), p->G);
        }
    }
    return DOCTORS_OK;
}

// choose the chunk: the option, or the largest balanced chunk that fits `budget` bytes
int choose_chunk(const doctors_problem* p, const doctors_solve_opts* o, size_t budget)
{
    int nprob = nprob_of(p);
    if (o && o->source_chunk > 0) return std::min(o->source_chunk, nprob);
    int best = 1;
    for (int c = 1; c <= nprob; ++c)
        if (make_plan(p, o, c).total <= budget) best = c;
    int nch = (nprob + best - 1) / best;
    return (nprob + nch - 1) / nch;
}

}  // namespace

// ------------------------------------------------------------------------------------------
extern "C" {

const char* doctors_version(void) { return "doctors-b200 0.1 (sm_100a)"; }

void doctors_abi_sizes(int* out_sizes)
{
    if (!out_sizes) return;
    out_sizes[0] = int(sizeof(doctors_source));
    out_sizes[1] = int(sizeof(doctors_solve_opts));
    out_sizes[2] = int(sizeof(doctors_solve_info));
}

int doctors_create_problem(int cuda_device, void* stream, doctors_problem** out)
{
    if (!out) return DOCTORS_INVALID_ARG;
    *out = nullptr;
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n <= 0 || cuda_device < 0 || cuda_device >= n) return DOCTORS_CUDA;
    if (cudaSetDevice(cuda_device) != cudaSuccess) return DOCTORS_CUDA;
    doctors_problem* p = new (std::nothrow) doctors_problem();
    if (!p) return DOCTORS_ALLOC;
    p->device = cuda_device;
    p->stream = static_cast<cudaStream_t>(stream);
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, cuda_device) != cudaSuccess) { delete p; return DOCTORS_CUDA; }
    p->num_sms = prop.multiProcessorCount;
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess || !fn) { delete p; return DOCTORS_CUDA; }
    p->encode = reinterpret_cast<decltype(p->encode)>(fn);
    *out = p;
    return DOCTORS_OK;
}

void doctors_destroy_problem(doctors_problem* p)
{
    if (!p) return;
    for (cudaEvent_t e : p->ev_pool) cudaEventDestroy(e);
    if (p->h_flag) cudaFreeHost(p->h_flag);
    delete p;
}

const char* doctors_last_error(const doctors_problem* p) { return p ? p->err.c_str() : "null handle"; }

int doctors_set_mesh_materials(doctors_problem* p, int nx, int ny, int nz, double dx, double dy, double dz,
                               const uint8_t* material_id, const float* density, int n_materials)
{
    if (!p) return DOCTORS_INVALID_ARG;
    if (nx <= 0 || ny <= 0 || nz <= 0) return fail(p, DOCTORS_INVALID_ARG, "mesh extents must be positive");
    if (!(dx > 0 && dy > 0 && dz > 0) || !std::isfinite(dx) || !std::isfinite(dy) || !std::isfinite(dz))
        return fail(p, DOCTORS_INVALID_ARG, "voxel pitch must be positive and finite");
    if (!material_id) return fail(p, DOCTORS_INVALID_ARG, "material_id is NULL");
    if (n_materials <= 0 || n_materials > kMaxMaterials)
        return fail(p, DOCTORS_INVALID_ARG, "n_materials must be 1..%d", kMaxMaterials);
    if ((long long)nx * ny * nz > (1LL << 30)) return fail(p, DOCTORS_INVALID_ARG, "mesh too large");
    size_t cells = size_t(nx) * ny * nz;
    for (size_t c = 0; c < cells; ++c) {
        if (material_id[c] >= n_materials) return fail(p, DOCTORS_INVALID_ARG, "material id %d >= n_materials at cell %zu", int(material_id[c]), c);
        if (density && !(density[c] >= 0.0f && std::isfinite(density[c])))
            return fail(p, DOCTORS_INVALID_ARG, "density must be finite and >= 0 (cell %zu)", c);
    }
    p->nx = nx; p->ny = ny; p->nz = nz; p->dx = dx; p->dy = dy; p->dz = dz;
    p->n_mat_mesh = n_materials;
    p->mat.assign(material_id, material_id + cells);
    if (density) p->rho.assign(density, density + cells); else p->rho.assign(cells, 1.0f);
    p->has_mesh = true;
    p->solved = false;
    ++p->inputs_version;
    return DOCTORS_OK;
}

int doctors_set_xs(doctors_problem* p, int n_materials, int n_groups, int pl_order, const double* sigma_t, const double* sigma_s)
{
    if (!p) return DOCTORS_INVALID_ARG;
    if (n_materials <= 0 || n_materials > kMaxMaterials) return fail(p, DOCTORS_INVALID_ARG, "n_materials must be 1..%d", kMaxMaterials);
    if (n_groups <= 0 || n_groups > 4096) return fail(p, DOCTORS_INVALID_ARG, "n_groups must be 1..4096");
    if (pl_order < 0 || pl_order > 3) return fail(p, DOCTORS_INVALID_ARG, "pl_order must be 0..3");
    if (!sigma_t || !sigma_s) return fail(p, DOCTORS_INVALID_ARG, "NULL table");
    const int G = n_groups, L = pl_order;
    for (int m = 0; m < n_materials; ++m)
        for (int g = 0; g < G; ++g)
            if (!(sigma_t[m * G + g] >= 0.0) || !std::isfinite(sigma_t[m * G + g]))
                return fail(p, DOCTORS_INVALID_ARG, "sigma_t[%d][%d] must be finite and >= 0", m, g);
    for (int m = 0; m < n_materials; ++m)
        for (int l = 0; l <= L; ++l)
            for (int gf = 0; gf < G; ++gf)
                for (int gt = 0; gt < G; ++gt) {
                    double v = sigma_s[((size_t(m) * (L + 1) + l) * G + gf) * G + gt];
                    if (!std::isfinite(v)) return fail(p, DOCTORS_INVALID_ARG, "sigma_s not finite");
                    if (gt < gf && v != 0.0)
                        return fail(p, DOCTORS_INVALID_ARG, "upscatter entry sigma_s[%d][%d][%d->%d] != 0 (downscatter only, PAPER.md:34)", m, l, gf, gt);
                }
    p->n_mat_xs = n_materials; p->G = G; p->L = L;
    p->sigt.assign(sigma_t, sigma_t + size_t(n_materials) * G);
    p->sigs.assign(sigma_s, sigma_s + size_t(n_materials) * (L + 1) * G * G);
    p->has_xs = true;
    p->solved = false;
    ++p->inputs_version;
    return DOCTORS_OK;
}

int doctors_set_quadrature(doctors_problem* p, int sn_order)
{
    if (!p) return DOCTORS_INVALID_ARG;
    std::vector<double> om, w;
    if (!level_symmetric(sn_order, om, w))
        return fail(p, DOCTORS_INVALID_ARG, "S_N order must be one of 2, 4, 6, 8, 12, 16");
    p->omega = om; p->w = w; p->ndir = int(w.size());
    p->has_quad = true;
    p->solved = false;
    ++p->inputs_version;
    return DOCTORS_OK;
}

int doctors_set_quadrature_points(doctors_problem* p, int n_dir, const double* omega_xyz, const double* w)
{
    if (!p) return DOCTORS_INVALID_ARG;
    if (n_dir <= 0 || n_dir % 8 != 0 || !omega_xyz || !w) return fail(p, DOCTORS_INVALID_ARG, "n_dir must be a positive multiple of 8");
    if (n_dir / 8 > 64) return fail(p, DOCTORS_INVALID_ARG, "at most 64 directions per octant");
    double sw = 0.0;
    std::vector<std::vector<int>> by_oct(8);
    const double pi = std::acos(-1.0);
    for (int n = 0; n < n_dir; ++n) {
        const double* o = omega_xyz + 3 * n;
        double nr = std::sqrt(o[0] * o[0] + o[1] * o[1] + o[2] * o[2]);
        if (std::fabs(nr - 1.0) > 1e-10) return fail(p, DOCTORS_INVALID_ARG, "direction %d is not a unit vector", n);
        if (o[0] == 0.0 || o[1] == 0.0 || o[2] == 0.0) return fail(p, DOCTORS_INVALID_ARG, "direction %d has a zero component", n);
        if (!(w[n] > 0.0)) return fail(p, DOCTORS_INVALID_ARG, "weight %d must be positive", n);
        sw += w[n];
        by_oct[(o[0] < 0 ? 1 : 0) | (o[1] < 0 ? 2 : 0) | (o[2] < 0 ? 4 : 0)].push_back(n);
    }
    if (std::fabs(sw - 4.0 * pi) > 1e-10 * 4.0 * pi) return fail(p, DOCTORS_INVALID_ARG, "weights sum to %.15g, not 4 pi", sw);
    for (int o = 0; o < 8; ++o)
        if (int(by_oct[o].size()) != n_dir / 8) return fail(p, DOCTORS_INVALID_ARG, "octant %d has %zu directions, expected %d", o, by_oct[o].size(), n_dir / 8);
    p->omega.clear(); p->w.clear();
    for (int o = 0; o < 8; ++o)
        for (int n : by_oct[o]) {
            p->omega.insert(p->omega.end(), omega_xyz + 3 * n, omega_xyz + 3 * n + 3);
            p->w.push_back(w[n]);
        }
    p->ndir = n_dir;
    p->has_quad = true;
    p->solved = false;
    ++p->inputs_version;
    return DOCTORS_OK;
}

int doctors_get_quadrature(const doctors_problem* p, int* n_dir, double* omega_xyz, double* w)
{
    if (!p || !n_dir) return DOCTORS_INVALID_ARG;
    if (!p->has_quad) return DOCTORS_BAD_STATE;
    *n_dir = p->ndir;
    if (omega_xyz) std::memcpy(omega_xyz, p->omega.data(), p->omega.size() * 8);
    if (w) std::memcpy(w, p->w.data(), p->w.size() * 8);
    return DOCTORS_OK;
}

int doctors_set_source(doctors_problem* p, int n_sources, const doctors_source* src, int mode)
{
    if (!p) return DOCTORS_INVALID_ARG;
    if (n_sources <= 0 || n_sources > 64 || !src) return fail(p, DOCTORS_INVALID_ARG, "n_sources must be 1..64");
    if (mode != 0 && mode != 1) return fail(p, DOCTORS_INVALID_ARG, "mode must be 0 or 1");
    if (!p->has_mesh || !p->has_xs) return fail(p, DOCTORS_BAD_STATE, "set the mesh and the cross sections before the source (array lengths)");
    std::vector<SourceHost> v(n_sources);
    const size_t cells = size_t(p->nx) * p->ny * p->nz;
    for (int s = 0; s < n_sources; ++s) {
        const doctors_source& S = src[s];
        SourceHost& H = v[s];
        H.kind = S.kind;
        if (S.kind == 0) {
            if (!S.volume) return fail(p, DOCTORS_INVALID_ARG, "source %d: volume is NULL", s);
            H.volume.assign(S.volume, S.volume + size_t(p->G) * cells);
            for (float f : H.volume) if (!std::isfinite(f)) return fail(p, DOCTORS_INVALID_ARG, "source %d: volume not finite", s);
        } else if (S.kind == 1 || S.kind == 2 || S.kind == 3) {
            if (!S.spectrum) return fail(p, DOCTORS_INVALID_ARG, "source %d: spectrum is NULL", s);
            H.spectrum.assign(S.spectrum, S.spectrum + p->G);
            for (int a = 0; a < 3; ++a) { H.pos[a] = S.pos[a]; H.axis[a] = S.axis[a]; }
            H.half = S.half_angle_rad;
            if (S.kind == 2 || S.kind == 3) {
                double an = std::sqrt(S.axis[0] * S.axis[0] + S.axis[1] * S.axis[1] + S.axis[2] * S.axis[2]);
                if (!(an > 0.0) || !(S.half_angle_rad > 0.0)) return fail(p, DOCTORS_INVALID_ARG, "source %d: cone / fan needs an axis and a half angle", s);
                for (int a = 0; a < 3; ++a) H.axis[a] = S.axis[a] / an;
            }
            if (S.kind == 3) {
                // normal of the fan plane: the part of `up` perpendicular to the axis
                const double ua = S.up[0] * H.axis[0] + S.up[1] * H.axis[1] + S.up[2] * H.axis[2];
                double nv[3], nn2 = 0.0;
                for (int a = 0; a < 3; ++a) { nv[a] = S.up[a] - ua * H.axis[a]; nn2 += nv[a] * nv[a]; }
                const double upn = S.up[0] * S.up[0] + S.up[1] * S.up[1] + S.up[2] * S.up[2];
                if (!(nn2 > 1e-24 * upn) || !(upn > 0.0)) return fail(p, DOCTORS_INVALID_ARG, "source %d: fan needs an up vector that is not parallel to its axis", s);
                if (!(S.half_angle2_rad > 0.0) || S.half_angle2_rad > 1.5707963267948968 || S.half_angle_rad > 3.1415926535897936)
                    return fail(p, DOCTORS_INVALID_ARG, "source %d: fan angles: 0 < half_angle <= pi, 0 < half_angle2 <= pi/2", s);
                for (int a = 0; a < 3; ++a) H.fan_n[a] = nv[a] / std::sqrt(nn2);
                H.half2 = S.half_angle2_rad;
            }
            // 1/R^2 singularity: a source on a cell centre
            const double d[3] = {p->dx, p->dy, p->dz};
            const int nn[3] = {p->nx, p->ny, p->nz};
            bool on_centre = true;
            for (int a = 0; a < 3; ++a) {
                double f = (S.pos[a] + 0.5 * nn[a] * d[a]) / d[a] - 0.5;      // fractional cell index
                double r = std::round(f);
                if (!(r >= 0 && r <= nn[a] - 1 && std::fabs(f - r) < 1e-9)) on_centre = false;
            }
            if (on_centre) return fail(p, DOCTORS_INVALID_ARG, "source %d sits on a cell centre (1/R^2 singularity)", s);
        } else {
            return fail(p, DOCTORS_INVALID_ARG, "source %d: unknown kind %d", s, S.kind);
        }
    }
    p->sources.swap(v);
    p->mode = mode;
    p->has_src = true;
    p->solved = false;
    ++p->inputs_version;
    return DOCTORS_OK;
}

int doctors_n_problems(const doctors_problem* p) { return p && p->has_src ? nprob_of(p) : 0; }

size_t doctors_workspace_bytes(doctors_problem* p, const doctors_solve_opts* opts)
{
    if (!p) return 0;
    if (check_ready(p) != DOCTORS_OK) return 0;
    size_t fr = 0, tot = 0;
    cudaSetDevice(p->device);
    if (cudaMemGetInfo(&fr, &tot) != cudaSuccess) { fail(p, DOCTORS_CUDA, "cudaMemGetInfo failed"); return 0; }
    int chunk = choose_chunk(p, opts, size_t(double(fr) * 0.85));
    return make_plan(p, opts, chunk).total;
}

int doctors_set_workspace(doctors_problem* p, void* device_ptr, size_t bytes)
{
    if (!p) return DOCTORS_INVALID_ARG;
    if (!device_ptr || (reinterpret_cast<uintptr_t>(device_ptr) & 255u)) return fail(p, DOCTORS_INVALID_ARG, "workspace must be non-NULL and 256-byte aligned");
    p->ws = device_ptr; p->ws_bytes = bytes;
    p->solved = false;
    ++p->inputs_version;
    return DOCTORS_OK;
}

long long doctors_wavefront_size(int nx, int ny, int nz, int S) { return wavefront_size(nx, ny, nz, S); }

int doctors_debug_schedule_dims(doctors_problem* p, const doctors_solve_opts* opts, int level, int dims[3])
{
    if (!p || !dims) return DOCTORS_INVALID_ARG;
    if (!p->has_mesh) return fail(p, DOCTORS_BAD_STATE, "mesh not set");
    if (level == 0) { dims[0] = p->nx; dims[1] = p->ny; dims[2] = p->nz; return DOCTORS_OK; }
    if (!p->has_xs || !p->has_quad) return fail(p, DOCTORS_BAD_STATE, "xs / quadrature not set (brick size depends on them)");
    int B[3];
    auto_brick((p->L + 1) * (p->L + 1), p->ndir / 8, p->nx, p->ny, p->nz, opts ? opts->brick : nullptr, wants_mma(opts, p->ndir / 8),
               face_bytes(opts && opts->closure == 1), B);
    if (level == 1) { for (int a = 0; a < 3; ++a) dims[a] = ((a == 0 ? p->nx : a == 1 ? p->ny : p->nz) + B[a] - 1) / B[a]; return DOCTORS_OK; }
    if (level == 2) { for (int a = 0; a < 3; ++a) dims[a] = B[a]; return DOCTORS_OK; }
    return fail(p, DOCTORS_INVALID_ARG, "level must be 0, 1 or 2");
}

int doctors_debug_get_schedule(doctors_problem* p, const doctors_solve_opts* opts, int octant, int level,
                               int32_t* plane_offset, int32_t* cell_of)
{
    if (!p || !plane_offset || !cell_of || octant < 0 || octant > 7) return DOCTORS_INVALID_ARG;
    int d[3];
    int rc = doctors_debug_schedule_dims(p, opts, level, d);
    if (rc != DOCTORS_OK) return rc;
    std::vector<int32_t> off, cells;
    subsweep_schedule(d[0], d[1], d[2], octant, off, cells);
    std::memcpy(plane_offset, off.data(), off.size() * 4);
    std::memcpy(cell_of, cells.data(), cells.size() * 4);
    return DOCTORS_OK;
}

int doctors_debug_get_tables(const doctors_problem* p, int pl_order, double* Mtab, double* Dtab)
{
    if (!p || pl_order < 0 || pl_order > 3 || !Mtab || !Dtab) return DOCTORS_INVALID_ARG;
    if (!p->has_quad) return DOCTORS_BAD_STATE;
    std::vector<double> M, D;
    projection_tables(pl_order, p->omega, p->w, M, D);
    std::memcpy(Mtab, M.data(), M.size() * 8);
    std::memcpy(Dtab, D.data(), D.size() * 8);
    return DOCTORS_OK;
}

int doctors_host_level_symmetric(int sn_order, double* omega_xyz, double* w)
{
    std::vector<double> om, ww;
    if (!omega_xyz || !w || !level_symmetric(sn_order, om, ww)) return DOCTORS_INVALID_ARG;
    std::memcpy(omega_xyz, om.data(), om.size() * 8);
    std::memcpy(w, ww.data(), ww.size() * 8);
    return DOCTORS_OK;
}

int doctors_host_schedule(int nx, int ny, int nz, int octant, int32_t* plane_offset, int32_t* cell_of)
{
    if (nx <= 0 || ny <= 0 || nz <= 0 || octant < 0 || octant > 7 || !plane_offset || !cell_of) return DOCTORS_INVALID_ARG;
    std::vector<int32_t> off, cells;
    subsweep_schedule(nx, ny, nz, octant, off, cells);
    std::memcpy(plane_offset, off.data(), off.size() * 4);
    std::memcpy(cell_of, cells.data(), cells.size() * 4);
    return DOCTORS_OK;
}

int doctors_host_pl_exceeds_quadrature(int pl_order, int n_dir, const double* omega_xyz, const double* w, double* defect)
{
    if (pl_order < 0 || pl_order > 3 || n_dir <= 0 || !omega_xyz || !w) return -1;
    std::vector<double> om(omega_xyz, omega_xyz + 3 * size_t(n_dir)), ww(w, w + n_dir);
    const double d = galerkin_defect(pl_order, om, ww);
    if (defect) *defect = d;
    return d > kGalerkinTol ? 1 : 0;
}

int doctors_host_projection_tables(int pl_order, int n_dir, const double* omega_xyz, const double* w, double* Mtab, double* Dtab)
{
    if (pl_order < 0 || pl_order > 3 || n_dir <= 0 || !omega_xyz || !w || !Mtab || !Dtab) return DOCTORS_INVALID_ARG;
    std::vector<double> om(omega_xyz, omega_xyz + 3 * size_t(n_dir)), ww(w, w + n_dir), M, D;
    projection_tables(pl_order, om, ww, M, D);
    std::memcpy(Mtab, M.data(), M.size() * 8);
    std::memcpy(Dtab, D.data(), D.size() * 8);
    return DOCTORS_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------
// solve
// ------------------------------------------------------------------------------------------
namespace {

__global__ void k_group_begin(ProbState* st, Control* ctl, const int* fixed_iters, int prob0, int n, int chunk, int G, int g, double* bal)
{
    int q = threadIdx.x;
    if (q >= n && q < chunk) st[q].done = 1;          // short last chunk: no such problem
    if (q < n) {
        ProbState s;
        s.max_diff_bits = 0u; s.max_phi_bits = 0u; s.iters = 0; s.done = 0;
        s.fixed = fixed_iters[(size_t)(prob0 + q) * G + g];
        s.hit_max = 0; s.resid = 0.0f; s.pad = 0;
        st[q] = s;
        bal[2 * q] = 0.0; bal[2 * q + 1] = 0.0;
    }
    if (q == 0) { ctl->ticket = 0u; ctl->all_done = 0; }
}

__global__ void k_group_end(const ProbState* st, const double* leak, const double* bal, GroupResult* res, int prob0, int n, int G, int g)
{
    int q = threadIdx.x;
    if (q < n) {
        GroupResult r;
        r.iters = st[q].iters; r.hit_max = st[q].hit_max; r.resid = st[q].resid; r.pad = 0.0f;
        r.leak = leak[q]; r.bal_src = bal[2 * q]; r.bal_col = bal[2 * q + 1];
        res[(size_t)(prob0 + q) * G + g] = r;
    }
}

// copy the scalar flux of the finished group into the retained array
__global__ void k_keep_phi0(long long cells_p, int g, int G, int NM, const float* __restrict__ phi_all,
                            float* __restrict__ phi0_all, int prob0)
{
    const int q = blockIdx.y;
    const float* src = phi_all + ((size_t)q * G + g) * NM * cells_p;
    float* dst = phi0_all + ((size_t)(prob0 + q) * G + g) * cells_p;
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < cells_p; c += (long long)gridDim.x * blockDim.x)
        dst[c] = src[c];
}

template <typename T>
T* at(doctors_problem* p, size_t off) { return reinterpret_cast<T*>(static_cast<char*>(p->ws) + off); }

int make_tensor_map(doctors_problem* p, CUtensorMap* tm, void* base, int rank, const cuuint64_t* dims,
                    const cuuint64_t* strides_bytes /*rank-1*/, const cuuint32_t* box,
                    CUtensorMapDataType dtype = CU_TENSOR_MAP_DATA_TYPE_FLOAT32)
{
    cuuint32_t es[5] = {1, 1, 1, 1, 1};
    CUresult r = p->encode(tm, dtype, cuuint32_t(rank), base, dims, strides_bytes, box, es,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                           CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(p, DOCTORS_CUDA, "cuTensorMapEncodeTiled failed (%d)", int(r));
    return DOCTORS_OK;
}

// the fixed-pitch instantiation (sweep_brick.cuh, PITCH = 640: 640-cell bricks, 10 directions per octant) exists for P3 with the
// FMA-loop projections: the shapes of configs 1, 2 and 4
constexpr int kFixedPitch = 640;        // 20 x 8 x 4 cells (the default brick)
constexpr int kFixedPitchLong = 768;    // 24 x 8 x 4 cells (opts.brick): fits three CTAs per SM with fp32 exchange faces; whole config-4 solve
                                        // 15.12 / 15.13 s per step against 15.15 / 15.17 s with the default brick (A/B): not worth a new default
template <int NM, int MT>
constexpr bool has_fixed_pitch() { return NM == 16 && MT == 0; }

template <int NM, bool FIX, int MT>
cudaError_t launch_brick(const SweepLaunch& S, cudaStream_t st)
{
    if constexpr (has_fixed_pitch<NM, MT>()) {
        if (S.bp.NCb == kFixedPitch && S.bp.M == 10) {
            k_sweep_brick<NM, FIX, MT, kFixedPitch><<<S.grid, 32 * S.bp.W, S.smem, st>>>(S.tmQ, S.tmPhi, S.bp);
            return cudaGetLastError();
        }
        if (S.bp.NCb == kFixedPitchLong && S.bp.M == 10) {
            k_sweep_brick<NM, FIX, MT, kFixedPitchLong><<<S.grid, 32 * S.bp.W, S.smem, st>>>(S.tmQ, S.tmPhi, S.bp);
            return cudaGetLastError();
        }
    }
    k_sweep_brick<NM, FIX, MT, 0><<<S.grid, 32 * S.bp.W, S.smem, st>>>(S.tmQ, S.tmPhi, S.bp);
    return cudaGetLastError();
}

template <int NM, bool FIX, int MT, int PITCH>
cudaError_t prep_one(size_t smem, int threads, int* max_ctas)
{
    cudaError_t e = cudaFuncSetAttribute(k_sweep_brick<NM, FIX, MT, PITCH>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem));
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(max_ctas, k_sweep_brick<NM, FIX, MT, PITCH>, threads, smem);
}

template <int NM, bool FIX, int MT>
cudaError_t prep_brick(int ncb, int m_oct, size_t smem, int threads, int* max_ctas)
{
    if constexpr (has_fixed_pitch<NM, MT>()) {
        if (ncb == kFixedPitch && m_oct == 10) return prep_one<NM, FIX, MT, kFixedPitch>(smem, threads, max_ctas);
        if (ncb == kFixedPitchLong && m_oct == 10) return prep_one<NM, FIX, MT, kFixedPitchLong>(smem, threads, max_ctas);
    }
    return prep_one<NM, FIX, MT, 0>(smem, threads, max_ctas);
}

// NM in {1, 4, 9, 16}; MT > 0 only with NM = 16 (projection_mtiles)
#define DISPATCH_ONE(NMc, FIXc, MTc, EXPR) { constexpr int NM = NMc; constexpr bool FIX = FIXc; constexpr int MT = MTc; EXPR; }
#define DISPATCH_NM(NMv, FIXc, MTv, EXPR)                                        \
    switch (NMv) {                                                               \
        case 1: DISPATCH_ONE(1, FIXc, 0, EXPR) break;                            \
        case 4: DISPATCH_ONE(4, FIXc, 0, EXPR) break;                            \
        case 9: DISPATCH_ONE(9, FIXc, 0, EXPR) break;                            \
        default:                                                                 \
            switch (MTv) {                                                       \
                case 1: DISPATCH_ONE(16, FIXc, 1, EXPR) break;                   \
                case 2: DISPATCH_ONE(16, FIXc, 2, EXPR) break;                   \
                case 3: DISPATCH_ONE(16, FIXc, 3, EXPR) break;                   \
                default: DISPATCH_ONE(16, FIXc, 0, EXPR) break;                  \
            }                                                                    \
            break;                                                               \
    }
#define DISPATCH_NM_FIX(NMv, FIXv, MTv, EXPR)                                    \
    do {                                                                         \
        if (FIXv) { DISPATCH_NM(NMv, true, MTv, EXPR) } else { DISPATCH_NM(NMv, false, MTv, EXPR) } \
    } while (0)

// TF32 rounding (round to nearest, ties away: what cvt.rna.tf32.f32 does) for the pre-split coefficient fragments
inline float tf32_rna(float v)
{
    uint32_t u; std::memcpy(&u, &v, 4);
    u = (u + 0x1000u) & 0xffffe000u;
    float r; std::memcpy(&r, &u, 4);
    return r;
}

// The per-octant table blobs of octtab_layout(): direction coefficients, leakage coefficients and the two
// projection tables (plain rows for the FFMA2 loops, pre-split mma A fragments for the tensor-core path).
std::vector<unsigned char> build_octtabs(int NM, int M, int MT, const std::vector<double>& dird, const std::vector<float4>& lkc,
                                         const std::vector<float>& Mt, const std::vector<float>& Dt)
{
    const OctTab T = octtab_layout(NM, M, MT);
    std::vector<unsigned char> blob(8 * T.total, 0);
    const int pitch = (NM + 3) / 4 * 4;
    for (int oc = 0; oc < 8; ++oc) {
        unsigned char* b = blob.data() + size_t(oc) * T.total;
        std::memcpy(b + T.dir, dird.data() + size_t(oc) * M * 4, size_t(M) * 32);
        std::memcpy(b + T.lk, lkc.data() + size_t(oc) * M, size_t(M) * 16);
        auto mt = [&](int n, int lm) { return n < M ? Mt[(size_t(oc) * M + n) * NM + lm] : 0.0f; };
        auto dt = [&](int n, int lm) { return n < M ? Dt[(size_t(oc) * M + n) * NM + lm] : 0.0f; };
        if (MT == 0) {
            float* m = reinterpret_cast<float*>(b + T.t0);
            float* d = reinterpret_cast<float*>(b + T.t2);
            for (int n = 0; n < M; ++n)
                for (int lm = 0; lm < NM; ++lm) { m[n * pitch + lm] = mt(n, lm); d[n * pitch + lm] = dt(n, lm); }
        } else {
            auto put = [](float* hi, float* lo, int lane, const float v[4]) {
                for (int r = 0; r < 4; ++r) { const float h = tf32_rna(v[r]); hi[lane * 4 + r] = h; lo[lane * 4 + r] = tf32_rna(v[r] - h); }
            };
            float* a0 = reinterpret_cast<float*>(b + T.t0);
            for (int t = 0; t < MT; ++t)
                for (int ks = 0; ks < 2; ++ks) {
                    float* hi = a0 + size_t((t * 2 + ks) * 2 + 0) * 128;
                    float* lo = a0 + size_t((t * 2 + ks) * 2 + 1) * 128;
                    for (int lane = 0; lane < 32; ++lane) {
                        const int g = lane >> 2, q = lane & 3;
                        const float v[4] = {mt(16 * t + g, 8 * ks + q), mt(16 * t + g + 8, 8 * ks + q), mt(16 * t + g, 8 * ks + q + 4), mt(16 * t + g + 8, 8 * ks + q + 4)};
                        put(hi, lo, lane, v);
                    }
                }
            float* a2 = reinterpret_cast<float*>(b + T.t2);
            for (int ks = 0; ks < 2 * MT; ++ks) {
                float* hi = a2 + size_t(ks * 2 + 0) * 128;
                float* lo = a2 + size_t(ks * 2 + 1) * 128;
                for (int lane = 0; lane < 32; ++lane) {
                    const int g = lane >> 2, q = lane & 3;
                    const float v[4] = {dt(8 * ks + q, g), dt(8 * ks + q, g + 8), dt(8 * ks + q + 4, g), dt(8 * ks + q + 4, g + 8)};
                    put(hi, lo, lane, v);
                }
            }
        }
    }
    return blob;
}

// Device-side set-up for one plan: inputs in brick-major order, tables, task list (a3), tensor maps.  Runs when an
// input, the workspace or a layout option changed (PrepKey); doctors_solve itself then only enqueues kernels.
int prepare(doctors_problem* p, const doctors_solve_opts& o, const Plan& P)
{
    cudaStream_t st = p->stream;
    const int NM = P.NM, G = P.G, L = P.L, M = P.M;
    const size_t cp = size_t(P.cells_p);
    const int nx = p->nx, ny = p->ny, nz = p->nz;
    MeshDev md;
    md.nx = nx; md.ny = ny; md.nz = nz; md.cells_p = P.cells_p;
    md.BX = P.B[0]; md.BY = P.B[1]; md.BZ = P.B[2]; md.gbx = P.gb[0]; md.gby = P.gb[1]; md.gbz = P.gb[2]; md.NCb = P.NCb;
    p->mesh_dev = md;
    md.dx = p->dx; md.dy = p->dy; md.dz = p->dz;
    md.x0 = 0.5 * p->dx - 0.5 * nx * p->dx; md.y0 = 0.5 * p->dy - 0.5 * ny * p->dy; md.z0 = 0.5 * p->dz - 0.5 * nz * p->dz;

    // ---- upload inputs and tables (brick-major order; padding cells: material 0, density 0) ----
    auto to_bricks = [&](const auto* dense, auto* bricked) {
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j) {
                const auto* row = dense + (size_t)nx * (j + (size_t)ny * k);
                for (int i = 0; i < nx; ++i) bricked[cell_index(md, i, j, k)] = row[i];
            }
    };
    {
        std::vector<uint8_t> hm(cp, 0);
        std::vector<float> hr(cp, 0.0f);
        to_bricks(p->mat.data(), hm.data());
        to_bricks(p->rho.data(), hr.data());
        CK(cudaMemcpyAsync(at<uint8_t>(p, P.o_mat), hm.data(), cp, cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(at<float>(p, P.o_rho), hr.data(), cp * 4, cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(at<uint8_t>(p, P.o_matd), p->mat.data(), p->mat.size(), cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(at<float>(p, P.o_rhod), p->rho.data(), p->rho.size() * 4, cudaMemcpyHostToDevice, st));
        CK(cudaStreamSynchronize(st));
    }
    std::vector<float> sigs_f(p->sigs.begin(), p->sigs.end());
    std::vector<double> spec(size_t(P.nsrc) * G, 0.0);
    std::vector<SourceDev> sdev(P.nsrc);
    {
        int slot = 0;
        for (int s = 0; s < P.nsrc; ++s) {
            const SourceHost& H = p->sources[s];
            SourceDev& D = sdev[s];
            D.kind = H.kind; D.vol_slot = -1;
            for (int a = 0; a < 3; ++a) { D.pos[a] = H.pos[a]; D.axis[a] = H.axis[a]; }
            D.cos_half = std::cos(H.half);
            for (int a = 0; a < 3; ++a) D.fan_n[a] = H.fan_n[a];
            D.sin_half2 = std::sin(H.half2);
            if (H.kind == 0) {
                D.vol_slot = slot;
                std::vector<float> hv(size_t(G) * cp, 0.0f);
                for (int g = 0; g < G; ++g) to_bricks(H.volume.data() + (size_t)g * nx * ny * nz, hv.data() + (size_t)g * cp);
                CK(cudaMemcpyAsync(at<float>(p, P.o_extvol) + (size_t)slot * G * cp, hv.data(), hv.size() * 4, cudaMemcpyHostToDevice, st));
                CK(cudaStreamSynchronize(st));
                ++slot;
            } else {
                for (int g = 0; g < G; ++g) spec[(size_t)s * G + g] = H.spectrum[g];
            }
        }
    }
    std::vector<double> Mt, Dt;
    projection_tables(L, p->omega, p->w, Mt, Dt);
    std::vector<float> Mt_f(Mt.begin(), Mt.end()), Dt_f(Dt.begin(), Dt.end());
    std::vector<float4> lkc(P.ndir);
    std::vector<double> dird(size_t(P.ndir) * 4);
    for (int n = 0; n < P.ndir; ++n) {
        double cx = 2.0 * std::fabs(p->omega[3 * n]) / p->dx, cy = 2.0 * std::fabs(p->omega[3 * n + 1]) / p->dy, cz = 2.0 * std::fabs(p->omega[3 * n + 2]) / p->dz;
        dird[4 * n] = cx; dird[4 * n + 1] = cy; dird[4 * n + 2] = cz; dird[4 * n + 3] = cx + cy + cz;
        lkc[n] = make_float4(float(p->w[n] * std::fabs(p->omega[3 * n]) * p->dy * p->dz),
                             float(p->w[n] * std::fabs(p->omega[3 * n + 1]) * p->dx * p->dz),
                             float(p->w[n] * std::fabs(p->omega[3 * n + 2]) * p->dx * p->dy), 0.0f);
    }
    CK(cudaMemcpyAsync(at<double>(p, P.o_sigt_hat), p->sigt.data(), p->sigt.size() * 8, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(at<float>(p, P.o_sigs), sigs_f.data(), sigs_f.size() * 4, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(at<double>(p, P.o_spec), spec.data(), spec.size() * 8, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(at<SourceDev>(p, P.o_srcs), sdev.data(), sdev.size() * sizeof(SourceDev), cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(at<float>(p, P.o_mtab), Mt_f.data(), Mt_f.size() * 4, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(at<float>(p, P.o_dtab), Dt_f.data(), Dt_f.size() * 4, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(at<double>(p, P.o_dird), dird.data(), dird.size() * 8, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(at<float4>(p, P.o_lk), lkc.data(), lkc.size() * 16, cudaMemcpyHostToDevice, st));

    // ---- schedules (a3) ----
    std::vector<uint2> tasks;
    std::vector<int>& oct_begin = p->oct_begin;
    oct_begin.assign(9, 0);
    std::vector<std::vector<int32_t>>& sched_off = p->sched_off;
    sched_off.assign(8, std::vector<int32_t>());
    SweepLaunch& SL = p->SL;
    int& ctas_per_sm = p->ctas_per_sm;
    ctas_per_sm = 0;
    int rc = DOCTORS_OK;
    if (P.sweep_mode == 0) {
        // level 2 (cells of a brick) needs no table: lane (j',k') at step s updates i' = s - j' - k' (Eq. 8)
        // level 1: bricks in sub-sweep order of the brick grid, per octant
        std::vector<std::vector<int32_t>> goff(8), gcell(8);
        for (int oc = 0; oc < 8; ++oc) subsweep_schedule(P.gb[0], P.gb[1], P.gb[2], oc, goff[oc], gcell[oc]);
        const int gplanes = P.gb[0] + P.gb[1] + P.gb[2] - 2;
        tasks.reserve(size_t(P.ntasks));
        auto push = [&](int q, int oc, int b) {
            int bi = b % P.gb[0], bj = (b / P.gb[0]) % P.gb[1], bk = b / (P.gb[0] * P.gb[1]);
            tasks.push_back(make_uint2(uint32_t(q) | uint32_t(oc) << 8, uint32_t(bi) | uint32_t(bj) << 10 | uint32_t(bk) << 20));
        };
        if (!P.deterministic) {
            // all problems and octants interleaved, brick sub-sweep S outermost
            for (int S = 0; S < gplanes; ++S)
                for (int q = 0; q < P.chunk; ++q)
                    for (int oc = 0; oc < 8; ++oc)
                        for (int t = goff[oc][S]; t < goff[oc][S + 1]; ++t) push(q, oc, gcell[oc][t]);
            oct_begin[0] = 0; oct_begin[1] = int(tasks.size());
        } else {
            for (int oc = 0; oc < 8; ++oc) {
                oct_begin[oc] = int(tasks.size());
                for (int S = 0; S < gplanes; ++S)
                    for (int q = 0; q < P.chunk; ++q)
                        for (int t = goff[oc][S]; t < goff[oc][S + 1]; ++t) push(q, oc, gcell[oc][t]);
            }
            oct_begin[8] = int(tasks.size());
        }
        CK(cudaMemcpyAsync(at<uint2>(p, P.o_tasks), tasks.data(), tasks.size() * sizeof(uint2), cudaMemcpyHostToDevice, st));
        CK(cudaMemsetAsync(at<unsigned>(p, P.o_flags), 0, size_t(P.chunk) * 8 * P.nbricks * 4, st));

        {
            // brick-major arrays: a brick's cells of one moment are tm_rows contiguous rows of tm_inner cells
            cuuint64_t d4[4] = {cuuint64_t(P.tm_inner), cuuint64_t(P.tm_rows) * P.nbricks, cuuint64_t(NM), cuuint64_t(P.chunk)};
            cuuint64_t s4[3] = {cuuint64_t(P.tm_inner) * 4, cuuint64_t(cp) * 4, cuuint64_t(cp) * NM * 4};
            cuuint32_t b4[4] = {cuuint32_t(P.tm_inner), cuuint32_t(P.tm_rows), cuuint32_t(NM), 1};
            rc = make_tensor_map(p, &SL.tmQ, at<float>(p, P.o_Q), 4, d4, s4, b4);
            if (rc != DOCTORS_OK) return rc;
            d4[3] = cuuint64_t(P.chunk) * G;
            rc = make_tensor_map(p, &SL.tmPhi, at<float>(p, P.o_phiall), 4, d4, s4, b4);
            if (rc != DOCTORS_OK) return rc;
        }
        {
            const std::vector<unsigned char> blob = build_octtabs(NM, M, P.MT, dird, lkc, Mt_f, Dt_f);
            CK(cudaMemcpyAsync(at<unsigned char>(p, P.o_octtab), blob.data(), blob.size(), cudaMemcpyHostToDevice, st));
            CK(cudaStreamSynchronize(st));
        }
        int max_ctas = 0;
        cudaError_t e = cudaSuccess;
        DISPATCH_NM_FIX(NM, o.closure == 1, P.MT, e = (prep_brick<NM, FIX, MT>(P.NCb, P.M, P.smem, 32 * P.W, &max_ctas)));
        if (e != cudaSuccess) return fail(p, DOCTORS_CUDA, "sweep kernel setup failed: %s (smem %zu)", cudaGetErrorString(e), P.smem);
        if (max_ctas < 1) return fail(p, DOCTORS_CUDA, "sweep kernel does not fit an SM (smem %zu)", P.smem);
        ctas_per_sm = o.ctas_per_sm > 0 ? std::min(o.ctas_per_sm, max_ctas) : max_ctas;
        SL.grid = p->num_sms * ctas_per_sm;
        SL.smem = P.smem;
        BrickParams& bp = SL.bp;
        bp.nx = nx; bp.ny = ny; bp.nz = nz;
        bp.BX = P.B[0]; bp.BY = P.B[1]; bp.BZ = P.B[2];
        bp.gbx = P.gb[0]; bp.gby = P.gb[1]; bp.gbz = P.gb[2];
        bp.M = M; bp.W = P.W; bp.g = 0; bp.Gs = G; bp.epoch = 0;
        bp.NCb = P.NCb; bp.cells_p = P.cells_p; bp.tm_rows = P.tm_rows; bp.nprob = P.chunk;
        bp.Q = at<float>(p, P.o_Q); bp.phi = at<float>(p, P.o_phiall); bp.sigt = at<double>(p, P.o_sigt);
        bp.octtab = at<unsigned char>(p, P.o_octtab);
        bp.tasks = at<uint2>(p, P.o_tasks);
        bp.ctl = at<Control>(p, P.o_ctl);
        bp.flags = at<unsigned>(p, P.o_flags);
        bp.faceX = at<char>(p, P.o_fx); bp.faceY = at<char>(p, P.o_fy); bp.faceZ = at<char>(p, P.o_fz);
        bp.dbg_plane = nullptr;
        {   // bulk async copies move multiples of 16 bytes
            const size_t q = 16 / P.fbytes;
            bp.bulk_faces = (P.face_x_n % q == 0 && P.face_y_n % q == 0 && P.face_z_n % q == 0) ? 1 : 0;
        }
        bp.state = at<ProbState>(p, P.o_state);
        bp.leak = at<double>(p, P.o_leak);
    } else {
        std::vector<int32_t> cells;
        for (int oc = 0; oc < 8; ++oc) {
            subsweep_schedule(nx, ny, nz, oc, sched_off[oc], cells);
            CK(cudaMemcpyAsync(at<int32_t>(p, P.o_sched) + (size_t)oc * nx * ny * nz, cells.data(), cells.size() * 4, cudaMemcpyHostToDevice, st));
            CK(cudaStreamSynchronize(st));
        }
    }
    CK(cudaStreamSynchronize(st));     // host staging vectors go out of scope here
    p->md = md;
    p->epoch = 0;                      // the flags were just cleared
    // Does the quadrature integrate the products Y_lm Y_l'm' exactly up to the P_L order set?  (Galerkin identity:
    // sum_n w_n Y_lm (2l'+1)/(4 pi) Y_l'm' = delta.  Level-symmetric sets: exact up to P1/P2/P3/P4 at S2/S4/S6/S8, >= P5 at
    // S12/S16, DESIGN.md App. A; a higher P_L still runs, the moments of the scattering source are then inconsistent.)
    p->pl_inexact = galerkin_defect(L, p->omega, p->w) > kGalerkinTol ? 1 : 0;
    return DOCTORS_OK;
}


}  // namespace

extern "C" int doctors_solve(doctors_problem* p, const doctors_solve_opts* opts_in, doctors_solve_info* info)
{
    if (!p) return DOCTORS_INVALID_ARG;
    int rc = check_ready(p);
    if (rc != DOCTORS_OK) return rc;
    doctors_solve_opts o;
    std::memset(&o, 0, sizeof o);
    if (opts_in) o = *opts_in;
    if (!(o.tol > 0.0)) o.tol = 1e-5;
    if (o.max_iters <= 0) o.max_iters = 100;
    const bool adaptive_window = o.check_window <= 0;   // first host read where the previous group stopped, then every sweep
    if (o.check_window <= 0) o.check_window = 12;
    if (o.closure != 0 && o.closure != 1) return fail(p, DOCTORS_INVALID_ARG, "closure must be 0 or 1");
    if (o.sweep_mode < 0 || o.sweep_mode > 1) return fail(p, DOCTORS_INVALID_ARG, "sweep_mode must be 0 or 1");
    if (o.brick[0] > 0 && (o.brick[0] % 4 != 0 || o.brick[0] > 64 || o.brick[1] <= 0 || o.brick[2] <= 0 || o.brick[1] * o.brick[2] > 32))
        return fail(p, DOCTORS_INVALID_ARG, "brick: brick[0] a multiple of 4 (<= 64), brick[1] * brick[2] <= 32 (the lanes of a warp)");
    if (!p->ws) return fail(p, DOCTORS_ALLOC, "no workspace set");
    CK(cudaSetDevice(p->device));
    cudaStream_t st = p->stream;

    const int chunk = choose_chunk(p, &o, p->ws_bytes);
    Plan P = make_plan(p, &o, chunk);
    if (P.total > p->ws_bytes)
        return fail(p, DOCTORS_ALLOC, "workspace too small: need %zu bytes (chunk %d), have %zu", P.total, P.chunk, p->ws_bytes);
    if (P.chunk > 255) return fail(p, DOCTORS_INVALID_ARG, "chunk too large");
    if (P.gb[0] > 1023 || P.gb[1] > 1023 || P.gb[2] > 1023) return fail(p, DOCTORS_INVALID_ARG, "brick grid too large");
    p->solved = false;
    p->plan = P;
    const int NM = P.NM, G = P.G, L = P.L, M = P.M;
    const size_t cp = size_t(P.cells_p);
    const int nx = p->nx, ny = p->ny, nz = p->nz;
    if (size_t(p->n_mat_xs) * (L + 1) * G * 4 > 200 * 1024)
        return fail(p, DOCTORS_INVALID_ARG, "scattering rows of one destination group (n_materials x (L+1) x G floats = %zu bytes) "
                    "do not fit the fixed-source kernel's shared memory (200 KB)", size_t(p->n_mat_xs) * (L + 1) * G * 4);

    PrepKey key;
    key.inputs_version = p->inputs_version; key.ws = p->ws; key.total = P.total; key.chunk = P.chunk;
    key.B[0] = P.B[0]; key.B[1] = P.B[1]; key.B[2] = P.B[2]; key.MT = P.MT; key.sweep_mode = P.sweep_mode;
    key.deterministic = P.deterministic; key.closure = o.closure; key.ctas_opt = o.ctas_per_sm;
    if (!p->prepared || !(p->prep_key == key)) {
        p->prepared = false;
        rc = prepare(p, o, P);
        if (rc != DOCTORS_OK) return rc;
        p->prepared = true;
        p->prep_key = key;
    }
    const MeshDev md = p->md;
    SweepLaunch& SL = p->SL;
    const std::vector<int>& oct_begin = p->oct_begin;
    const std::vector<std::vector<int32_t>>& sched_off = p->sched_off;
    const int ctas_per_sm = p->ctas_per_sm;
    std::vector<int> fixed_h(size_t(P.nprob) * G, 0);
    if (o.fixed_iters) std::copy(o.fixed_iters, o.fixed_iters + fixed_h.size(), fixed_h.begin());
    CK(cudaMemcpyAsync(at<int>(p, P.o_fixediters), fixed_h.data(), fixed_h.size() * 4, cudaMemcpyHostToDevice, st));
    CK(cudaStreamSynchronize(st));           // fixed_h is pageable: the copy is staged, but do not rely on it

    // ---- events: a pool owned by the handle; every sweep launch is timed, however long the solve ----
    p->ev_used = 0;
    cudaError_t ev_err = cudaSuccess;
    auto next_event = [&]() -> cudaEvent_t {
        if (p->ev_used == p->ev_pool.size()) {
            cudaEvent_t e = nullptr;
            cudaError_t ce = cudaEventCreate(&e);
            if (ce != cudaSuccess) { ev_err = ce; return nullptr; }
            p->ev_pool.push_back(e);
        }
        return p->ev_pool[p->ev_used++];
    };
#define NEXT_EVENT(var)                                                                                      \
    cudaEvent_t var = next_event();                                                                          \
    if (!var) return fail(p, DOCTORS_CUDA, "cudaEventCreate failed: %s", cudaGetErrorString(ev_err))
    NEXT_EVENT(ev_total0); NEXT_EVENT(ev_total1); NEXT_EVENT(ev_a); NEXT_EVENT(ev_b);
    std::vector<cudaEvent_t> sweep_ev, fixed_ev, iter_ev;       // pairs (the events themselves live in the pool)
    double ms_ray = 0.0;
    unsigned long long sweep_launches = 0, kernel_launches = 0, updates = 0;
    unsigned& epoch = p->epoch;
    if (!p->h_flag) CK(cudaMallocHost(&p->h_flag, 64));
    int* h_flag = p->h_flag;
    bool not_converged = false;
    const unsigned cblocks = unsigned((P.cells_p + 255) / 256);
    const int red_blocks = int(std::min<long long>((P.cells_p + 255) / 256, 4LL * p->num_sms));
    {
        // the fixed-source kernel stages the scattering rows of the destination group in shared memory
        const size_t need = size_t(p->n_mat_xs) * (L + 1) * G * 4;
        if (need > 48 * 1024) {
            cudaError_t e = cudaSuccess;
            switch (NM) {
                case 1: e = cudaFuncSetAttribute(k_fixed_source<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(need)); break;
                case 4: e = cudaFuncSetAttribute(k_fixed_source<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(need)); break;
                case 9: e = cudaFuncSetAttribute(k_fixed_source<9>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(need)); break;
                default: e = cudaFuncSetAttribute(k_fixed_source<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(need)); break;
            }
            if (e != cudaSuccess) return fail(p, DOCTORS_CUDA, "fixed-source kernel setup failed: %s", cudaGetErrorString(e));
        }
    }

    NvtxRange nvtx_solve("doctors_solve");
    CK(cudaEventRecord(ev_total0, st));
    for (int ch = 0; ch < P.nchunks; ++ch) {
        const int prob0 = ch * P.chunk;
        const int nq = std::min(P.chunk, P.nprob - prob0);           // problems in this chunk
        const int src0 = P.mode == 0 ? prob0 : 0;
        const int nsrc_c = P.mode == 0 ? nq : P.nsrc;
        float* phi_u_c = at<float>(p, P.o_phiu) + (size_t)src0 * G * cp;

        // a1: uncollided flux of the chunk's sources
        {
        NvtxRange nvtx_ray("a1 raytrace");
        CK(cudaEventRecord(ev_a, st));
        k_raytrace<<<dim3(unsigned((P.cells_p + kRayThreads - 1) / kRayThreads), nsrc_c), kRayThreads, 0, st>>>(
            md, at<uint8_t>(p, P.o_matd), at<float>(p, P.o_rhod), at<SourceDev>(p, P.o_srcs), src0,
            at<double>(p, P.o_sigt_hat), at<double>(p, P.o_spec), p->n_mat_xs, G, phi_u_c);
        CK(cudaGetLastError());
        ++kernel_launches;
        CK(cudaEventRecord(ev_b, st));
        CK(cudaEventSynchronize(ev_b));
        { float ms = 0; cudaEventElapsedTime(&ms, ev_a, ev_b); ms_ray += ms; }
        }

        int prev_group_iters = 0;                                 // sweeps the previous group of this chunk needed
        for (int g = 0; g < G; ++g) {
            NvtxRange nvtx_group("group: a2 fixed source + a6 source iteration (a3-a5 sweeps)");
            k_group_begin<<<1, 256, 0, st>>>(at<ProbState>(p, P.o_state), at<Control>(p, P.o_ctl), at<int>(p, P.o_fixediters),
                                              prob0, nq, P.chunk, G, g, at<double>(p, P.o_bal));
            k_sigt<<<cblocks, 256, 0, st>>>(md, at<uint8_t>(p, P.o_mat), at<float>(p, P.o_rho), at<double>(p, P.o_sigt_hat), G, g, at<double>(p, P.o_sigt));
            NEXT_EVENT(f0); NEXT_EVENT(f1);
            fixed_ev.push_back(f0); fixed_ev.push_back(f1);
            CK(cudaEventRecord(f0, st));
            {
                size_t sm = size_t(p->n_mat_xs) * (L + 1) * (g + 1) * 4;
#define LAUNCH_FIXED(NMv)                                                                                          \
    k_fixed_source<NMv><<<dim3(cblocks, nq), 256, sm, st>>>(md, at<uint8_t>(p, P.o_mat), at<float>(p, P.o_rho),       \
        at<float>(p, P.o_sigs), p->n_mat_xs, L, G, g, at<SourceDev>(p, P.o_srcs), src0, nsrc_c, P.mode, phi_u_c,   \
        at<float>(p, P.o_extvol), at<float>(p, P.o_phiall), at<float>(p, P.o_fixed))
                switch (NM) { case 1: LAUNCH_FIXED(1); break; case 4: LAUNCH_FIXED(4); break; case 9: LAUNCH_FIXED(9); break; default: LAUNCH_FIXED(16); }
#undef LAUNCH_FIXED
            }
            CK(cudaGetLastError());
            CK(cudaEventRecord(f1, st));
            kernel_launches += 3;

            // fixed replay: every problem of the chunk has a count -> enqueue exactly max count, no host read
            int max_fixed = 0; bool all_fixed = true;
            for (int q = 0; q < nq; ++q) {
                int f = fixed_h[(size_t)(prob0 + q) * G + g];
                if (f <= 0) all_fixed = false;
                max_fixed = std::max(max_fixed, f);
            }
            const int limit = all_fixed ? max_fixed : std::max(o.max_iters, max_fixed);
            NEXT_EVENT(i0); NEXT_EVENT(i1);
            iter_ev.push_back(i0); iter_ev.push_back(i1);
            CK(cudaEventRecord(i0, st));
            int k = 0;
            while (k < limit) {
                int batch = all_fixed ? limit : std::min(o.check_window, limit - k);
                if (!all_fixed && adaptive_window)
                    batch = std::min(limit - k, k == 0 ? (prev_group_iters > 1 ? prev_group_iters - 1 : std::min(o.check_window, 6)) : 1);
                for (int b = 0; b < batch; ++b, ++k) {
#define LAUNCH_UPDATE(NMv)                                                                                          \
    k_update<NMv><<<dim3((cblocks + 3) / 4, nq), 256, 0, st>>>(md, at<uint8_t>(p, P.o_mat), at<float>(p, P.o_rho), at<float>(p, P.o_sigs), \
        p->n_mat_xs, L, G, g, G, k == 0 ? 1 : 0, at<float>(p, P.o_fixed), at<float>(p, P.o_phiall), at<float>(p, P.o_Q),          \
        at<float>(p, P.o_phi0old), at<ProbState>(p, P.o_state), at<Control>(p, P.o_ctl), at<double>(p, P.o_leak))
                    switch (NM) { case 1: LAUNCH_UPDATE(1); break; case 4: LAUNCH_UPDATE(4); break; case 9: LAUNCH_UPDATE(9); break; default: LAUNCH_UPDATE(16); }
#undef LAUNCH_UPDATE
                    ++kernel_launches;
                    NEXT_EVENT(s0); NEXT_EVENT(s1);
                    sweep_ev.push_back(s0); sweep_ev.push_back(s1);
                    CK(cudaEventRecord(s0, st));
                    if (P.sweep_mode == 0) {
                        SL.bp.g = g;
                        const int nl = P.deterministic ? 8 : 1;
                        for (int l = 0; l < nl; ++l) {
                            SL.bp.epoch = ++epoch;
                            SL.bp.counter_slot = l;
                            SL.bp.task_begin = oct_begin[l];
                            // the list is built for P.chunk problems; a short last chunk marks the missing
                            // problems done (k_group_begin), so their tasks are skipped
                            SL.bp.ntasks = oct_begin[l + 1] - oct_begin[l];
                            cudaError_t e;
                            DISPATCH_NM_FIX(NM, o.closure == 1, P.MT, e = (launch_brick<NM, FIX, MT>(SL, st)));
                            if (e != cudaSuccess) return fail(p, DOCTORS_CUDA, "sweep launch failed: %s", cudaGetErrorString(e));
                            ++sweep_launches; ++kernel_launches;
                        }
                    } else {
                        const int planes = nx + ny + nz - 2;
                        for (int oc = 0; oc < 8; ++oc)
                            for (int S = 0; S < planes; ++S) {
                                const int cnt = sched_off[oc][S + 1] - sched_off[oc][S];
                                const int32_t* cl = at<int32_t>(p, P.o_sched) + (size_t)oc * nx * ny * nz + sched_off[oc][S];
#define LAUNCH_SUB(NMv, FIXv)                                                                                        \
    k_subsweep<NMv, FIXv><<<dim3((cnt + 127) / 128, nq), 128, 0, st>>>(md, cl, cnt, oc, M, at<float>(p, P.o_mtab),      \
        at<float>(p, P.o_dtab), at<double>(p, P.o_dird), at<float4>(p, P.o_lk), at<double>(p, P.o_sigt), at<float>(p, P.o_Q), \
        at<float>(p, P.o_phiall), g, G, at<double>(p, P.o_ox), at<double>(p, P.o_oy), at<double>(p, P.o_oz),            \
        at<ProbState>(p, P.o_state), at<double>(p, P.o_leak))
                                if (o.closure == 1) { switch (NM) { case 1: LAUNCH_SUB(1, true); break; case 4: LAUNCH_SUB(4, true); break; case 9: LAUNCH_SUB(9, true); break; default: LAUNCH_SUB(16, true); } }
                                else { switch (NM) { case 1: LAUNCH_SUB(1, false); break; case 4: LAUNCH_SUB(4, false); break; case 9: LAUNCH_SUB(9, false); break; default: LAUNCH_SUB(16, false); } }
#undef LAUNCH_SUB
                                ++sweep_launches; ++kernel_launches;
                            }
                    }
                    CK(cudaEventRecord(s1, st));
                    k_check<<<dim3(red_blocks, nq), 256, 0, st>>>(md, g, G, NM, at<float>(p, P.o_phiall), at<float>(p, P.o_phi0old),
                                                                   at<ProbState>(p, P.o_state), at<Control>(p, P.o_ctl), nq, float(o.tol), o.max_iters);
                    ++kernel_launches;
                }
                CK(cudaGetLastError());
                if (all_fixed) break;
                CK(cudaMemcpyAsync(h_flag, &at<Control>(p, P.o_ctl)->all_done, 4, cudaMemcpyDeviceToHost, st));
                CK(cudaStreamSynchronize(st));
                if (*h_flag) break;
            }
            prev_group_iters = k;
            CK(cudaEventRecord(i1, st));
            k_balance<<<dim3(red_blocks, nq), 256, 0, st>>>(md, g, G, NM, at<float>(p, P.o_phiall), at<float>(p, P.o_Q), at<double>(p, P.o_sigt),
                                                             p->dx * p->dy * p->dz, at<double>(p, P.o_bal));
            k_group_end<<<1, 256, 0, st>>>(at<ProbState>(p, P.o_state), at<double>(p, P.o_leak), at<double>(p, P.o_bal),
                                            at<GroupResult>(p, P.o_results), prob0, nq, G, g);
            k_keep_phi0<<<dim3(red_blocks, nq), 256, 0, st>>>(P.cells_p, g, G, NM, at<float>(p, P.o_phiall), at<float>(p, P.o_phi0all), prob0);
            kernel_launches += 3;
            CK(cudaGetLastError());
        }
        p->last_chunk_first = prob0;
        p->last_chunk_count = nq;
    }
    CK(cudaEventRecord(ev_total1, st));
    CK(cudaStreamSynchronize(st));
    CK(cudaGetLastError());

    // ---- results ----
    std::vector<GroupResult> res(size_t(P.nprob) * G);
    CK(cudaMemcpy(res.data(), at<GroupResult>(p, P.o_results), res.size() * sizeof(GroupResult), cudaMemcpyDeviceToHost));
    for (size_t t = 0; t < res.size(); ++t) {
        updates += (unsigned long long)res[t].iters * (unsigned long long)nx * ny * nz * P.ndir;
        if (res[t].hit_max) not_converged = true;
    }
    if (info) {
        for (size_t t = 0; t < res.size(); ++t) {
            if (info->iters) info->iters[t] = res[t].iters;
            if (info->residual) info->residual[t] = res[t].resid;
            if (info->balance) { info->balance[3 * t] = res[t].bal_src; info->balance[3 * t + 1] = res[t].bal_col; info->balance[3 * t + 2] = res[t].leak; }
        }
        float ms = 0;
        cudaEventElapsedTime(&ms, ev_total0, ev_total1); info->ms_total = ms;
        info->ms_raytrace = ms_ray;
        double acc = 0; for (size_t e = 0; e + 1 < sweep_ev.size(); e += 2) { cudaEventElapsedTime(&ms, sweep_ev[e], sweep_ev[e + 1]); acc += ms; }
        info->ms_sweep = acc;
        acc = 0; for (size_t e = 0; e + 1 < fixed_ev.size(); e += 2) { cudaEventElapsedTime(&ms, fixed_ev[e], fixed_ev[e + 1]); acc += ms; }
        info->ms_fixed_source = acc;
        acc = 0; for (size_t e = 0; e + 1 < iter_ev.size(); e += 2) { cudaEventElapsedTime(&ms, iter_ev[e], iter_ev[e + 1]); acc += ms; }
        info->ms_iterate = acc;
        info->updates = updates;
        info->sweep_launches = sweep_launches;
        info->kernel_launches = kernel_launches;
        info->n_chunks = P.nchunks;
        info->brick[0] = P.B[0]; info->brick[1] = P.B[1]; info->brick[2] = P.B[2];
        info->ctas_per_sm = ctas_per_sm;
        info->projection_mtiles = P.sweep_mode == 0 ? P.MT : 0;
        info->sweep_kernel = o.sweep_mode == 1 ? 1 : 0;
        info->timed_sweeps = (unsigned long long)(sweep_ev.size() / 2);
        info->pl_exceeds_quadrature = p->pl_inexact;
    }
#undef NEXT_EVENT
    p->solved = true;
    if (not_converged) { p->err = "some (problem, group) stopped at max_iters"; return DOCTORS_NOT_CONVERGED; }
    return DOCTORS_OK;
}

namespace {
// brick-major device fields -> dense [field][nz][ny][nx] rows (host or device destination)
int copy_rows_out(doctors_problem* p, const float* src, float* out, int out_is_device, int n_fields)
{
    const Plan& P = p->plan;
    const size_t n = size_t(p->nx) * p->ny * p->nz * n_fields;
    float* dst = out_is_device ? out : at<float>(p, P.o_scratch);
    const int blocks = int(std::min<size_t>((n + 255) / 256, size_t(16) * p->num_sms));
    k_unbrick<<<blocks, 256, 0, p->stream>>>(p->mesh_dev, src, dst, n_fields);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && !out_is_device) e = cudaMemcpyAsync(out, dst, n * 4, cudaMemcpyDeviceToHost, p->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
    if (e != cudaSuccess) return fail(p, DOCTORS_CUDA, "copy out failed: %s", cudaGetErrorString(e));
    return DOCTORS_OK;
}
}  // namespace

// Test hook: run the product sweep kernel (its debug instantiation) on ONE full brick of the given
// shape and octant and report, per cell, the wavefront step at which the kernel updated it.
extern "C" int doctors_debug_device_brick_steps(doctors_problem* p, int bx, int by, int bz, int octant, int32_t* step_of_cell)
{
    if (!p || !step_of_cell || octant < 0 || octant > 7) return DOCTORS_INVALID_ARG;
    if (bx <= 0 || bx % 4 != 0 || bx > 64 || by <= 0 || bz <= 0 || by * bz > 32)
        return fail(p, DOCTORS_INVALID_ARG, "brick: bx a multiple of 4 (<= 64), by * bz <= 32");
    CK(cudaSetDevice(p->device));
    const int NC = bx * by * bz;
    const size_t smem = brick_smem_layout(1, bx, by, bz, 1, 0, face_bytes(false)).total;
    // scratch: Q, phi (float), sigt (double), faces (double), table blobs, control
    struct Scratch { float* Q; float* phi; double* sig; double* face; unsigned char* tab; uint2* task;
                     unsigned* flags; Control* ctl; ProbState* st; double* leak; int* planes; } S;
    const size_t nface = size_t(by) * bz + size_t(bx) * bz + size_t(bx) * by;
    const OctTab T = octtab_layout(1, 1, 0);
    char* base = nullptr;
    const size_t bytes = 8192 + size_t(NC) * (4 + 4 + 8 + 4) + 256 + nface * 8 * 2 + 8 * T.total;
    CK(cudaMalloc(&base, bytes));
    CK(cudaMemset(base, 0, bytes));
    size_t off = 0;
    auto take = [&](size_t n) { char* r = base + off; off = align_up(off + n, 256); return r; };
    S.Q = (float*)take(size_t(NC) * 4); S.phi = (float*)take(size_t(NC) * 4); S.sig = (double*)take(size_t(NC) * 8);
    S.planes = (int*)take(size_t(NC) * 4 + 4); S.face = (double*)take(nface * 8);
    S.tab = (unsigned char*)take(8 * T.total); S.task = (uint2*)take(16);
    S.flags = (unsigned*)take(64); S.ctl = (Control*)take(sizeof(Control)); S.st = (ProbState*)take(sizeof(ProbState)); S.leak = (double*)take(8);
    if (off > bytes) { cudaFree(base); return fail(p, DOCTORS_ALLOC, "debug scratch too small"); }
    const uint2 task = make_uint2(uint32_t(octant) << 8, 0u);
    {
        // one direction per octant with coefficients (1, 1, 1, sum 3) and unit projection tables
        std::vector<double> dd(32); for (int i = 0; i < 32; ++i) dd[i] = (i % 4 == 3) ? 3.0 : 1.0;
        std::vector<float4> lk(8, make_float4(0.f, 0.f, 0.f, 0.f));
        std::vector<float> one(8, 1.0f);
        const std::vector<unsigned char> blob = build_octtabs(1, 1, 0, dd, lk, one, one);
        cudaMemcpy(S.tab, blob.data(), blob.size(), cudaMemcpyHostToDevice);
    }
    cudaMemcpy(S.task, &task, sizeof task, cudaMemcpyHostToDevice);
    SweepLaunch SL;
    int rows = 1;
    while ((NC / 4) % rows != 0 || NC / rows > 256) ++rows;
    {
        const int inner = NC / rows;
        cuuint64_t d4[4] = {cuuint64_t(inner), cuuint64_t(rows), 1, 1};
        cuuint64_t s4[3] = {cuuint64_t(inner) * 4, cuuint64_t(NC) * 4, cuuint64_t(NC) * 4};
        cuuint32_t b4[4] = {cuuint32_t(inner), cuuint32_t(rows), 1, 1};
        int rc = make_tensor_map(p, &SL.tmQ, S.Q, 4, d4, s4, b4);
        if (rc == DOCTORS_OK) rc = make_tensor_map(p, &SL.tmPhi, S.phi, 4, d4, s4, b4);
        if (rc != DOCTORS_OK) { cudaFree(base); return rc; }
    }
    BrickParams& bp = SL.bp;
    std::memset(&bp, 0, sizeof bp);
    bp.tm_rows = rows; bp.nprob = 1;
    bp.nx = bx; bp.ny = by; bp.nz = bz; bp.BX = bx; bp.BY = by; bp.BZ = bz; bp.gbx = bp.gby = bp.gbz = 1;
    bp.M = 1; bp.W = 1; bp.g = 0; bp.Gs = 1; bp.epoch = 1; bp.task_begin = 0; bp.ntasks = 1; bp.counter_slot = 0;
    bp.NCb = NC; bp.cells_p = NC; bp.Q = S.Q; bp.phi = S.phi; bp.sigt = S.sig; bp.octtab = S.tab;
    bp.tasks = S.task; bp.ctl = S.ctl; bp.flags = S.flags;
    bp.faceX = S.face; bp.faceY = S.face + size_t(by) * bz; bp.faceZ = S.face + size_t(by) * bz + size_t(bx) * bz;   // element offsets (fp64 faces: closure 0)
    bp.state = S.st; bp.leak = S.leak;
    bp.dbg_plane = S.planes;
    cudaError_t e = cudaFuncSetAttribute(k_sweep_brick<1, false, 0, 0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem));
    if (e == cudaSuccess) {
        k_sweep_brick<1, false, 0, 0, true><<<1, 32, smem, p->stream>>>(SL.tmQ, SL.tmPhi, bp);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
    std::vector<int32_t> stored(size_t(NC) + 1, -1);
    if (e == cudaSuccess) e = cudaMemcpy(stored.data(), S.planes, size_t(NC) * 4 + 4, cudaMemcpyDeviceToHost);
    cudaFree(base);
    if (e == cudaSuccess && stored[size_t(NC)] != 0)
        return fail(p, DOCTORS_CUDA, "wavefront loop: %d shared-memory addresses outside the CTA's allocation (brick %d x %d x %d, octant %d)",
                    int(stored[size_t(NC)]), bx, by, bz, octant);
    for (int lk = 0; lk < bz; ++lk)                             // storage order inside a brick (y fastest) -> documented order
        for (int lj = 0; lj < by; ++lj)
            for (int li = 0; li < bx; ++li) step_of_cell[li + bx * (lj + by * lk)] = stored[size_t(lj + by * (li + bx * lk))];
    if (e != cudaSuccess) return fail(p, DOCTORS_CUDA, "debug brick launch failed: %s", cudaGetErrorString(e));
    return DOCTORS_OK;
}

extern "C" int doctors_get_flux_moments(doctors_problem* p, int problem, int group, int l_max, float* out, int out_is_device)
{
    if (!p || !out) return DOCTORS_INVALID_ARG;
    if (!p->solved) return fail(p, DOCTORS_BAD_STATE, "no successful solve yet");
    const Plan& P = p->plan;
    if (problem < 0 || problem >= P.nprob || group < 0 || group >= P.G || l_max < 0 || l_max > P.L)
        return fail(p, DOCTORS_INVALID_ARG, "bad problem / group / l_max");
    cudaSetDevice(p->device);
    const size_t cp = size_t(P.cells_p);
    if (l_max == 0) {
        const float* src = at<float>(p, P.o_phi0all) + ((size_t)problem * P.G + group) * cp;
        return copy_rows_out(p, src, out, out_is_device, 1);
    }
    if (problem < p->last_chunk_first || problem >= p->last_chunk_first + p->last_chunk_count)
        return fail(p, DOCTORS_NOT_RETAINED, "moments l > 0 of problem %d were overwritten by a later chunk", problem);
    const int q = problem - p->last_chunk_first;
    const int nmo = (l_max + 1) * (l_max + 1);
    const float* src = at<float>(p, P.o_phiall) + ((size_t)q * P.G + group) * P.NM * cp;
    return copy_rows_out(p, src, out, out_is_device, nmo);
}

extern "C" int doctors_get_response(doctors_problem* p, int problem, const double* response, int include_uncollided,
                                    float* out, int out_is_device)
{
    if (!p || !out || !response) return DOCTORS_INVALID_ARG;
    if (!p->solved) return fail(p, DOCTORS_BAD_STATE, "no successful solve yet");
    const Plan& P = p->plan;
    if (problem < 0 || problem >= P.nprob) return fail(p, DOCTORS_INVALID_ARG, "bad problem");
    cudaSetDevice(p->device);
    const size_t cp = size_t(P.cells_p), n = size_t(p->nx) * p->ny * p->nz;
    double* d_resp = at<double>(p, P.o_resp);
    cudaError_t e = cudaMemcpyAsync(d_resp, response, size_t(P.G) * 8, cudaMemcpyHostToDevice, p->stream);
    // mode 0: problem q is source q; mode 1: the one problem sums all sources
    const int src0 = P.mode == 0 ? problem : 0, nsrc = P.mode == 0 ? 1 : P.nsrc;
    bool any_unc = false;
    for (int s_ = src0; s_ < src0 + nsrc; ++s_) if (p->sources[size_t(s_)].kind != 0) any_unc = true;
    float* dst = out_is_device ? out : at<float>(p, P.o_scratch);
    const int blocks = int(std::min<size_t>((n + 255) / 256, size_t(16) * p->num_sms));
    if (e == cudaSuccess) {
        k_response<<<blocks, 256, 0, p->stream>>>(p->mesh_dev, P.G, d_resp, at<float>(p, P.o_phi0all) + (size_t)problem * P.G * cp,
                                                   (include_uncollided && any_unc) ? at<float>(p, P.o_phiu) : nullptr, src0, nsrc, dst);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess && !out_is_device) e = cudaMemcpyAsync(out, dst, n * 4, cudaMemcpyDeviceToHost, p->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
    if (e != cudaSuccess) return fail(p, DOCTORS_CUDA, "response failed: %s", cudaGetErrorString(e));
    return DOCTORS_OK;
}

extern "C" int doctors_get_uncollided_flux(doctors_problem* p, int source, int group, float* out, int out_is_device)
{
    if (!p || !out) return DOCTORS_INVALID_ARG;
    if (!p->solved) return fail(p, DOCTORS_BAD_STATE, "no successful solve yet");
    const Plan& P = p->plan;
    if (source < 0 || source >= P.nsrc || group < 0 || group >= P.G) return fail(p, DOCTORS_INVALID_ARG, "bad source / group");
    cudaSetDevice(p->device);
    const float* src = at<float>(p, P.o_phiu) + ((size_t)source * P.G + group) * size_t(P.cells_p);
    return copy_rows_out(p, src, out, out_is_device, 1);
}

// ------------------------------------------------------------------------------------------
// Allocation-free entry point: the convergence measure of row a6 (reading R8),
//   delta = max_c |phi_new(c) - phi_old(c)| / max_c |phi_new(c)|   per problem,
// for callers that may not allocate (CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
// It is a variant of k_check: the same max-reduction over the cells, but the cross-block scratch (per-block partial
// maxima, last-block tickets) lives in a file-scope __device__ array instead of the caller's workspace, and the result
// goes to a caller buffer instead of the solver's ProbState.  Every GPU that loads the library holds the array
// (sizeof(DeltaScratch) = 33,024 bytes) until the process exits.
//   - ALL calls on a device share the array: calls that overlap on the GPU (two streams, two handles) race.
//   - The array keeps the last call's contents; what must start at zero (the tickets) is cleared by a memset node on
//     the caller's stream before every launch, the partial maxima are fully rewritten before they are read.
//   - No cudaMalloc / cudaFree / allocating library routine is called.  The FIRST call per device looks the array's
//     device address up (cudaGetSymbolAddress: in host code the array's name is only a stand-in, not a device pointer);
//     make that first call outside a graph capture.
// ------------------------------------------------------------------------------------------
namespace {

constexpr int kDeltaBlocks = 64;            // blocks per problem (grid-stride over the cells)
constexpr int kDeltaMaxProblems = 64;       // stated maximum: problems per call (doctors_set_source takes at most 64 sources)
constexpr int kDeltaMaxDevices = 64;

struct DeltaScratch {
    float part[kDeltaMaxProblems][kDeltaBlocks][2];   // per block: max |new - old|, max |new|
    unsigned ticket[kDeltaMaxProblems];               // blocks of the problem that have finished (must start at 0)
};

static __device__ __align__(256) unsigned char g_delta_scratch[sizeof(DeltaScratch)];

__global__ void __launch_bounds__(256)
k_delta_static(DeltaScratch* S, const float* __restrict__ phi_new, const float* __restrict__ phi_old, long long n,
               long long stride, float* __restrict__ out /*[n_problems][3]: delta, max |new - old|, max |new|*/)
{
    const int p = blockIdx.y;
    const float* a = phi_new + (size_t)p * stride;
    const float* b = phi_old + (size_t)p * stride;
    float md = 0.0f, mp = 0.0f;
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < n; c += (long long)gridDim.x * blockDim.x) {
        const float v = a[c];
        md = fmaxf(md, fabsf(v - b[c]));
        mp = fmaxf(mp, fabsf(v));
        if (!(v == v) || !(b[c] == b[c])) md = INFINITY;            // NaN: visible in the result (fmaxf would drop it)
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
        S->part[p][blockIdx.x][0] = md;
        S->part[p][blockIdx.x][1] = mp;
        __threadfence();
        s_last = atomicAdd(&S->ticket[p], 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (s_last && threadIdx.x == 0) {
        __threadfence();
        float d = 0.0f, m = 0.0f;
        for (unsigned blk = 0; blk < gridDim.x; ++blk) {              // fixed order; max is order-independent anyway
            d = fmaxf(d, __ldcg(&S->part[p][blk][0]));
            m = fmaxf(m, __ldcg(&S->part[p][blk][1]));
        }
        out[3 * p] = m == 0.0f ? 0.0f : (float)((double)d / (double)m);   // as k_check: no source reaches the group -> 0
        out[3 * p + 1] = d;
        out[3 * p + 2] = m;
    }
}

}  // namespace

extern "C" int doctors_convergence_delta_no_alloc(doctors_problem* p, const float* device_phi_new, const float* device_phi_old,
                                                  long long n_cells, long long problem_stride, int n_problems, float* device_out)
{
    if (!p) return DOCTORS_INVALID_ARG;
    if (!device_phi_new || !device_phi_old || !device_out) return fail(p, DOCTORS_INVALID_ARG, "NULL device pointer");
    if (n_problems < 1 || n_problems > kDeltaMaxProblems)
        return fail(p, DOCTORS_INVALID_ARG, "n_problems = %d: the static scratch of doctors_convergence_delta_no_alloc holds at most %d problems per call",
                    n_problems, kDeltaMaxProblems);
    if (n_cells < 1 || n_cells > (1LL << 40)) return fail(p, DOCTORS_INVALID_ARG, "n_cells must be 1 .. 2^40");
    if (problem_stride < n_cells && n_problems > 1) return fail(p, DOCTORS_INVALID_ARG, "problem_stride must be >= n_cells");
    if (p->device < 0 || p->device >= kDeltaMaxDevices) return fail(p, DOCTORS_INVALID_ARG, "device ordinal beyond %d", kDeltaMaxDevices - 1);
    CK(cudaSetDevice(p->device));
    // set-up, once per device, with that device current: the device address of the static scratch
    static DeltaScratch* scratch_of[kDeltaMaxDevices] = {};
    if (!scratch_of[p->device]) {
        void* ptr = nullptr;
        CK(cudaGetSymbolAddress(&ptr, g_delta_scratch));
        if (!ptr) return fail(p, DOCTORS_CUDA, "cudaGetSymbolAddress returned a null address");
        scratch_of[p->device] = static_cast<DeltaScratch*>(ptr);
    }
    DeltaScratch* S = scratch_of[p->device];
    CK(cudaMemsetAsync(S->ticket, 0, sizeof S->ticket, p->stream));   // shared, keeps the last call's contents: tickets start at zero
    const unsigned bx = unsigned(std::min<long long>(kDeltaBlocks, (n_cells + 255) / 256));
    k_delta_static<<<dim3(bx, unsigned(n_problems)), 256, 0, p->stream>>>(S, device_phi_new, device_phi_old, n_cells, problem_stride, device_out);
    CK(cudaGetLastError());
    return DOCTORS_OK;
}
