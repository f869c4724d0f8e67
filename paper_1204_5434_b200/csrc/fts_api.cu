// fts_api.cu — host side of the C-ABI library declared in include/fts.h: context, workspace layout,
// host-built tables (S1), the launch schedule of one RQM4 contour step (S3-S5), Q (S7), densities (S6),
// field updates (S8-S9) and operators (S10).  No device allocation happens here: everything lives in
// the caller's workspace.  No CPU fallback: every arithmetic step of the path is a kernel in fts_kernels.cuh.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/fts.h"
#include "fts_kernels.cuh"
#include "fts_march.cuh"
#include "fts_march2.cuh"
#include "fts_plane.cuh"

namespace fts {

static const long double kPiL = 3.14159265358979323846264338327950288L;

struct DimTables { void* tab[2]; void* tw; void* tw2; double* k2; };

struct Ctx {
    int g[3]; double L[3]; int Ns; fts_params P; fts_precision prec;
    size_t M; int nprop, nspecies, jA; size_t esz;
    char* ws; size_t ws_bytes;
    // workspace carve-up
    DimTables dim[3];
    double *cA, *cB, *scal, *kacc; double2* partial;
    signed char* seg;             // device: species per contour segment
    std::vector<int> blk_species, blk_steps;      // chain architecture: blocks from the s = 0 end (fts_set_blocks)
    void *f0, *f1, *e4[2], *F[2], *H[2], *q[2], *phi[2], *G[2], *acc[2][2];
    int keep, nslots;             // slice store: slices 0..keep at slot s, the last slice of a march at slot keep + 1 (fts_march.cuh)
    bool have_fields, have_prop, have_phi; int marched;
    bool ops_entry;               // the last call was fts_cl_step: Q, the slices and the field sums of the fields it STARTED from are still there
    // march schedule (fts_march.cuh)
    Phase* phases;            // device: persistent template at [0], the four per-launch templates at [MARCH_MAXPH * (1..4)]
    unsigned* counters;       // device: completion counters, then ticket and error flag
    size_t counters_bytes;
    int persistent, planes, nchunks, lag, nph, tickets_per_round, cnt[4], sms, occ;
    // options (fts_set_option; no environment variables are read)
    struct { int march; long long slab_bytes; int lag, interleave, tz, skew, real_fields, graph, plane, tline; } opt;
    // per-phase launch mode: the whole march (4 launches per step) captured once as a CUDA graph and replayed (launch-bound loop)
    struct MarchGraph { cudaGraphExec_t exec; int nsteps; long long kernels; } graphs[2];
    int ngraphs; cudaStream_t cap_stream;
    int packed;                   // N1 real-field fast path active: one march of z = q + i q+ (fts_march.cuh); nprop is then 1
    // TMA march for large cubic grids (fts_march2.cuh)
    int v2, v2_lag, v2_skew, v2_occ;
    March2Maps maps;
    std::string err;
};

static uint64_t g_launches = 0;      // kernels launched by this library since it was loaded (bench.py's gpu_launches)

static size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }
enum { MARCH_MAXCHUNKS = 64 };
static int counters_per_step(const int g[3]) { const int a = 2 + 2 * MARCH_MAXCHUNKS, b = 2 + 2 * g[0]; return a > b ? a : b; }

struct Layout {          // the single place that decides where things live in the workspace
    size_t off_tab[3][2], off_tw[3], off_tw2[3], off_k2[3], off_cA, off_cB, off_seg, off_scal, off_kacc, off_partial, off_phases, off_counters, counters_bytes;
    size_t off_f[2], off_e4[2], off_F[2], off_H[2], off_q[2], off_phi[2], off_G[2], off_acc[2][2], total; int keep, nslots;
};
static Layout make_layout(const int g[3], int Ns, int model, size_t esz, int store_both) {
    Layout Lo; size_t o = 0;
    const size_t M = (size_t)g[0] * g[1] * g[2], field = align_up(M * esz);
    const int nprop = model == FTS_MODEL_DIBLOCK ? 2 : 1;
    for (int d = 0; d < 3; ++d) {
        for (int h = 0; h < 2; ++h) { Lo.off_tab[d][h] = o; o += align_up((size_t)g[d] * esz / 2); }
        Lo.off_tw[d] = o; o += align_up((size_t)g[d] * esz);
        Lo.off_tw2[d] = o; o += align_up((size_t)g[d] * esz);
        Lo.off_k2[d] = o; o += align_up((size_t)g[d] * sizeof(double));
    }
    Lo.off_cA = o; o += align_up((size_t)(Ns + 1) * sizeof(double));
    Lo.off_cB = o; o += align_up((size_t)(Ns + 1) * sizeof(double));
    Lo.off_seg = o; o += align_up((size_t)Ns + 1);
    Lo.off_scal = o; o += align_up(64 * sizeof(double));
    Lo.off_kacc = o; o += align_up((size_t)(Ns + 1) * 2 * sizeof(double));
    Lo.off_partial = o; o += align_up(1024 * sizeof(double2));
    Lo.off_phases = o; o += align_up(5 * MARCH_MAXPH * sizeof(Phase));
    Lo.counters_bytes = align_up((size_t)2 * (Ns + 1) * counters_per_step(g) * sizeof(unsigned)) + 256;
    Lo.off_counters = o; o += Lo.counters_bytes;
    for (int i = 0; i < 2; ++i) { Lo.off_f[i] = o; o += field; }
    for (int i = 0; i < 2; ++i) { Lo.off_e4[i] = o; o += field; }
    for (int i = 0; i < 2; ++i) { Lo.off_F[i] = o; o += (i < nprop) ? field : 0; }
    for (int i = 0; i < 2; ++i) { Lo.off_H[i] = o; o += (i < nprop) ? field : 0; }
    for (int i = 0; i < 2; ++i) { Lo.off_phi[i] = o; o += field; }
    for (int i = 0; i < 2; ++i) { Lo.off_G[i] = o; o += field; }
    for (int b = 0; b < 2; ++b)
        for (int a = 0; a < 2; ++a) { Lo.off_acc[b][a] = o; o += (b < nprop && a < nprop) ? field : 0; }      // density sums [propagator][species]
    // contour-slice store: meet-in-the-middle keeps slices 0..Ns/2 and the last one per propagator,
    // store_both keeps all Ns + 1 (needed for Pi)
    Lo.keep = store_both ? Ns : Ns / 2;
    Lo.nslots = store_both ? Ns + 1 : Ns / 2 + 2;
    for (int i = 0; i < 2; ++i) { Lo.off_q[i] = o; o += (i < nprop) ? align_up((size_t)Lo.nslots * M * esz) : 0; }
    Lo.total = o;
    return Lo;
}

static int ept_of(int N) { return N == 1 ? 1 : ((N == 16 || N >= 128) ? 16 : 8); }     // must match the launch_*_n switches
static bool pow2_ok(int n) { return n == 1 || (n >= 8 && n <= 256 && (n & (n - 1)) == 0); }

// 1-D and 2-D problems (Fig. 1) are grids with dimensions of 1.  A dimension of 1 does not affect the
// memory layout ([ix][iy][iz], z contiguous), so internally the ones are moved to the front: (N,1,1) -> (1,1,N),
// (Nx,Ny,1) -> (1,Nx,Ny).  The kernels then see pencils of length 1 along x (and y) - the identity - and a real z.
static void squeeze_grid(const int grid[3], const double* cell, int g[3], double L[3]) {
    int n = 2;
    for (int d = 2; d >= 0; --d) if (grid[d] != 1) { g[n] = grid[d]; L[n] = cell ? cell[d] : 1.0; --n; }
    for (int d = 2; d >= 0 && n >= 0; --d) if (grid[d] == 1) { g[n] = 1; L[n] = cell ? cell[d] : 1.0; --n; }
}

static fts_status validate(const int grid[3], const double* cell, int Ns, const fts_params* P, int prec) {
    if (!grid || !P) return FTS_EINVAL;
    if (prec != FTS_F64 && prec != FTS_F32) return FTS_EINVAL;
    if (Ns < 2 || P->model < 0 || P->model > 2) return FTS_EINVAL;
    for (int d = 0; d < 3; ++d) {
        if (grid[d] < 1) return FTS_EINVAL;
        if (cell && !(cell[d] > 0)) return FTS_EINVAL;
    }
    if (P->model == FTS_MODEL_DIBLOCK) {
        const double x = P->fA * Ns; const long j = std::lround(x);
        if (std::fabs(x - (double)j) > 1e-9 || j <= 0 || j >= Ns) return FTS_EINVAL;     // reading A-4
        if ((j & 1) || ((Ns - j) & 1)) return FTS_EINVAL;                                  // reading A-5 (Simpson)
        if (!(P->chiN > 0)) return FTS_EINVAL;
    } else if (Ns & 1) return FTS_EINVAL;
    for (int d = 0; d < 3; ++d) if (!pow2_ok(grid[d])) return FTS_EUNSUPPORTED;
    if (grid[0] == 1 && grid[1] == 1 && grid[2] == 1) return FTS_EUNSUPPORTED;
    return FTS_OK;
}

#define CK(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess) {                                                                   \
            c->err = std::string(#call) + ": " + cudaGetErrorString(e_);                           \
            return FTS_ECUDA;                                                                      \
        }                                                                                          \
    } while (0)

// ------------------------------------------------------------------------------------------------
// pass launch: picks the instantiation for (precision, pencil length, strided or contiguous)
// ------------------------------------------------------------------------------------------------
template <class T, int N, int EPT, int TZ>
static cudaError_t launch_pass_inst(const PassArgs& A, int njobs, cudaStream_t st) {
    typedef PassCfg<T, N, EPT, TZ> Cfg;
    // set on every launch: the attribute is per device, and a process may drive several GPUs
    cudaError_t e = cudaFuncSetAttribute(pass_kernel<T, N, EPT, TZ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM);
    if (e != cudaSuccess) return e;
    dim3 grid((A.ntiles + Cfg::GPB - 1) / Cfg::GPB, njobs);
    pass_kernel<T, N, EPT, TZ><<<grid, Cfg::THREADS, Cfg::SMEM, st>>>(A);
    g_launches += 1;
    return cudaGetLastError();
}
template <class T, int TZ>
static cudaError_t launch_pass_n(int N, const PassArgs& A, int njobs, cudaStream_t st) {
    switch (N) {
        case 1: return launch_pass_inst<T, 1, 1, TZ>(A, njobs, st);
        case 8: return launch_pass_inst<T, 8, 8, TZ>(A, njobs, st);
        case 16: return launch_pass_inst<T, 16, 16, TZ>(A, njobs, st);
        case 32: return launch_pass_inst<T, 32, 8, TZ>(A, njobs, st);
        case 64: return launch_pass_inst<T, 64, 8, TZ>(A, njobs, st);
        case 128: return launch_pass_inst<T, 128, 16, TZ>(A, njobs, st);
        case 256: return launch_pass_inst<T, 256, 16, TZ>(A, njobs, st);
    }
    return cudaErrorInvalidValue;
}
template <class T> constexpr int tz_of() { return 128 / (2 * (int)sizeof(T)); }   // 128-byte rows

// dim: 0 = x, 1 = y (strided pencils, tiles of TZ consecutive z), 2 = z (contiguous pencils)
template <class T>
static cudaError_t launch_pass(const Ctx* c, int dim, PassArgs A, int njobs, cudaStream_t st) {
    const int Nx = c->g[0], Ny = c->g[1], Nz = c->g[2];
    A.tw = c->dim[dim].tw;
    A.k2x = c->dim[0].k2; A.k2y = c->dim[1].k2; A.k2z = c->dim[2].k2; A.Nz = Nz;
    A.invN = 1.0 / (double)c->g[dim];
    if (dim == 2) {
        A.pstride = 1; A.outer_stride = 0; A.tiles_inner = 1; A.ntiles = Nx * Ny;
        return launch_pass_n<T, 0>(Nz, A, njobs, st);
    }
    constexpr int TZ = tz_of<T>();
    const int tz = Nz < TZ ? 8 : TZ;                       // complex64 with Nz = 8: 64-byte rows
    if (dim == 0) { A.pstride = Ny * Nz; A.outer_stride = 0; A.tiles_inner = Ny * Nz / tz; A.ntiles = Ny * Nz / tz; }
    else { A.pstride = Nz; A.outer_stride = Ny * Nz; A.tiles_inner = Nz / tz; A.ntiles = Nx * Nz / tz; }
    if (tz == TZ) return launch_pass_n<T, TZ>(c->g[dim], A, njobs, st);
    return launch_pass_n<T, 8>(c->g[dim], A, njobs, st);
}

static Job mkjob(const void* in, void* out, int op) { Job j; j.in = in; j.out = out; j.op = op; return j; }

static int ew_blocks(size_t M) { size_t b = (M + 255) / 256; return (int)(b < 148 * 16 ? b : 148 * 16); }

template <class T, int OP>
static cudaError_t reduce(const Ctx* c, const void* a, const void* b, double p, double scale, double* out_dev, cudaStream_t st, const int* poison = nullptr) {
    const int M = (int)c->M;
    int nb = (M + RED_THREADS - 1) / RED_THREADS; if (nb > RED_BLOCKS) nb = RED_BLOCKS;
    reduce_partial_kernel<T, OP><<<nb, RED_THREADS, 0, st>>>((const cplx<T>*)a, (const cplx<T>*)b, M, p, c->partial);
    reduce_final_kernel<OP><<<1, 1024, 0, st>>>(c->partial, nb, scale, out_dev, poison);
    g_launches += 2;
    return cudaGetLastError();
}

// scalar slots in c->scal
enum { S_Q = 0, S_H = 2, S_RP = 4, S_RM = 6, S_SQ = 8, S_Q0 = 10 };

// ------------------------------------------------------------------------------------------------
// S2-S7: the march (fts_march.cuh).  Cubic grids: one persistent launch for the whole march, work items in a
// fixed ticket order with completion counters.  Other grids: the same kernel, one launch per phase kind and
// round (stream order replaces the counters), instantiated for that dimension's pencil length.
// ------------------------------------------------------------------------------------------------
struct MarchInfo { int threads, gpb_s, gpb_c; size_t smem; };

template <class T, int N, int EPT, int TZ>
static cudaError_t launch_march_inst(const MarchArgs& A, int grid, bool query, MarchInfo* info, int* occ, cudaStream_t st) {
    typedef MarchCfg<T, N, EPT, TZ> Cfg;
    if (info) { info->threads = Cfg::LAUNCH; info->gpb_s = Cfg::GPB_S; info->gpb_c = Cfg::GPB_C; info->smem = Cfg::SMEM; }
    if (query && !occ) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(march_kernel<T, N, EPT, TZ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM);
    if (e != cudaSuccess) return e;
    if (occ) {
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ, march_kernel<T, N, EPT, TZ>, Cfg::LAUNCH, Cfg::SMEM);
        if (e != cudaSuccess) return e;
    }
    if (query) return cudaSuccess;
    if (A.ticket) march_kernel<T, N, EPT, TZ><<<grid, Cfg::LAUNCH, Cfg::SMEM, st>>>(A);
    else {                                                 // per-phase launch: programmatic dependent launch (see the kernel's prologue)
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(grid); cfg.blockDim = dim3(Cfg::LAUNCH); cfg.dynamicSmemBytes = Cfg::SMEM; cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization; at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        e = cudaLaunchKernelEx(&cfg, march_kernel<T, N, EPT, TZ>, A);
        if (e != cudaSuccess) return e;
    }
    g_launches += 1;
    return cudaGetLastError();
}
template <class T, int TZ>
static cudaError_t launch_march_n(int N, const MarchArgs& A, int grid, bool query, MarchInfo* info, int* occ, cudaStream_t st) {
    switch (N) {
        case 1: return launch_march_inst<T, 1, 1, TZ>(A, grid, query, info, occ, st);
        case 8: return launch_march_inst<T, 8, 8, TZ>(A, grid, query, info, occ, st);
        case 16: return launch_march_inst<T, 16, 16, TZ>(A, grid, query, info, occ, st);
        case 32: return launch_march_inst<T, 32, 8, TZ>(A, grid, query, info, occ, st);
        case 64: return launch_march_inst<T, 64, 8, TZ>(A, grid, query, info, occ, st);
        case 128: return launch_march_inst<T, 128, 16, TZ>(A, grid, query, info, occ, st);
        case 256: return launch_march_inst<T, 256, 16, TZ>(A, grid, query, info, occ, st);
    }
    return cudaErrorInvalidValue;
}
// tz: pencils per strided tile = complex elements per 128-byte row, or 8 when Nz is shorter than that (complex64, Nz = 8)
// Pencils per strided tile: one 128-byte row (8 complex128, 16 complex64) unless z is shorter.  complex64 at pencil
// length 256 uses 64-byte rows instead: its 128-byte-row CTA (256 + 32 threads) is register-starved (measured: 681 vs 736 us per step at 256^3).
template <class T> static int tz_used(const Ctx* c) {
    const int full = tz_of<T>();
    if (c->opt.tz == 8) return 8;
    if (c->opt.tz == 16 && c->g[2] >= full) return full;
    if (sizeof(T) == 4 && (c->g[0] >= 256 || c->g[1] >= 256 || c->g[2] >= 256)) return 8;
    return c->g[2] >= full ? full : 8;
}
template <class T>
static cudaError_t launch_march(const Ctx* c, int N, const MarchArgs& A, int grid, bool query, MarchInfo* info, int* occ, cudaStream_t st) {
    if (tz_used<T>(c) == tz_of<T>()) return launch_march_n<T, tz_of<T>()>(N, A, grid, query, info, occ, st);
    return launch_march_n<T, 8>(N, A, grid, query, info, occ, st);
}

static int ceil_div(int a, int b) { return (a + b - 1) / b; }

static Phase mkphase(int first, int kind, int b, int prev, int chunk) {
    Phase p; p.first = first; p.chunk = (short)chunk; p.kind = (signed char)kind; p.prop_off = (signed char)(b | (prev << 1));
    return p;
}

// Ticket counts of one T phase and of one slab's Y1 / Z / Y2 phase for the instantiation `mi`.
static void phase_counts(const Ctx* c, const MarchInfo& mx, const MarchInfo& my, const MarchInfo& mz, int tz, int planes, int cnt[4]) {
    const int Ny = c->g[1], Nz = c->g[2];
    cnt[PH_T] = ceil_div(Ny * Nz / tz, mx.gpb_s);
    cnt[PH_Y1] = 2 * ceil_div(planes * (Nz / tz), my.gpb_s);
    cnt[PH_Z] = 2 * ceil_div(planes * Ny, mz.gpb_c);
    cnt[PH_Y2] = ceil_div(planes * (Nz / tz), my.gpb_s);
}

// Round template of the persistent march.  Two propagators:  T(q,j) | U(q+,j-1) & U(q,j) | T(q+,j)  so that every
// whole-field dependency (T -> U of the same step, U -> T of the next) is separated by the other propagator's items.
// U = the slabs' Y1, Z, Y2 phases software-pipelined `lag` slabs apart; the two propagators' U phases alternate
// (FTS_INTERLEAVE=0: one block per propagator).
static std::vector<Phase> make_template(int nprop, int nchunks, int lag, bool interleave, const int cnt[4], int* tickets) {
    std::vector<Phase> v; int first = 0;
    auto add = [&](int kind, int b, int prev, int chunk) { v.push_back(mkphase(first, kind, b, prev, chunk)); first += cnt[kind]; };
    auto ublock = [&](int b, int prev) {
        for (int i = 0; i < nchunks + 2 * lag; ++i) {
            if (i < nchunks) add(PH_Y1, b, prev, i);
            if (i - lag >= 0 && i - lag < nchunks) add(PH_Z, b, prev, i - lag);
            if (i - 2 * lag >= 0 && i - 2 * lag < nchunks) add(PH_Y2, b, prev, i - 2 * lag);
        }
    };
    add(PH_T, 0, 0, 0);
    if (nprop == 2 && interleave) {
        // alternate the two propagators phase by phase, so that a phase and the one it waits for are always separated by a
        // phase of the other propagator: no head-of-line blocking in ticket order (measured: -16 % at 64^3, -14 % at 128^3 fp32)
        for (int i = 0; i < nchunks + 2 * lag; ++i) {
            if (i < nchunks) { add(PH_Y1, 1, 1, i); add(PH_Y1, 0, 0, i); }
            if (i - lag >= 0 && i - lag < nchunks) { add(PH_Z, 1, 1, i - lag); add(PH_Z, 0, 0, i - lag); }
            if (i - 2 * lag >= 0 && i - 2 * lag < nchunks) { add(PH_Y2, 1, 1, i - 2 * lag); add(PH_Y2, 0, 0, i - 2 * lag); }
        }
    } else {
        if (nprop == 2) ublock(1, 1);
        ublock(0, 0);
    }
    if (nprop == 2) add(PH_T, 1, 0, 0);
    *tickets = first;
    return v;
}

// Boltzmann-factor fields: per species, or (packed mode) per species pair; the pair fields 2, 3 live in the second propagator's
// F and H, which the packed march does not use
static const void* e4_field(const Ctx* c, int i) { return i < 2 ? c->e4[i] : (c->packed ? (i == 2 ? c->F[1] : c->H[1]) : c->e4[i - 2]); }

static DensArgs dens_args(const Ctx* c, int nsteps) {
    DensArgs D;
    for (int b = 0; b < 2; ++b) for (int a = 0; a < 2; ++a) D.acc[b][a] = c->acc[b][a];
    // accumulate inside the march only with the meet-in-the-middle store; a full store is summed by density_store_kernel afterwards
    D.cA = c->cA; D.cB = c->cB; D.on = nsteps == c->Ns && c->keep != c->Ns; D.keep = c->keep; D.half = c->Ns / 2;
    return D;
}

template <class T>
static void fill_march_args(const Ctx* c, MarchArgs& A, int nsteps) {
    std::memset(&A, 0, sizeof A);
    for (int b = 0; b < 2; ++b) { A.q[b] = c->q[b]; A.F[b] = c->F[b]; A.H[b] = c->H[b]; }
    for (int i = 0; i < 4; ++i) A.e4[i] = e4_field(c, i);
    A.nprop = c->nprop; A.packed = c->packed;
    for (int d = 0; d < 3; ++d) { A.tab[d][0] = c->dim[d].tab[0]; A.tab[d][1] = c->dim[d].tab[1]; A.tw[d] = c->dim[d].tw; A.g[d] = c->g[d]; }
    A.M = (long long)c->M; A.Ns = c->Ns; A.jA = c->jA; A.nspecies = c->nspecies; A.nsteps = nsteps; A.seg = c->seg;
    A.done = c->counters; A.err = (int*)((char*)c->counters + c->counters_bytes - 128);
    A.dens = dens_args(c, nsteps);
}

// Decide the schedule once per context (needs the device: occupancy, SM count) and upload the templates.
template <class T>
static fts_status plan_march(Ctx* c) {
    const int Nx = c->g[0], Ny = c->g[1], Nz = c->g[2], tz = tz_used<T>(c);
    MarchArgs A; fill_march_args<T>(c, A, 0);
    MarchInfo mi[3];
    for (int d = 0; d < 3; ++d) CK(launch_march<T>(c, c->g[d], A, 0, true, &mi[d], nullptr, 0));
    int dev = 0; CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&c->sms, cudaDevAttrMultiProcessorCount, dev));
    c->persistent = (Nx == Ny && Ny == Nz) && c->opt.march != FTS_MARCH_LAUNCH;
    // Automatic choice for small cubic grids, from measurement (B200, Ns = 100, per diblock solve): the per-phase launches,
    // replayed as one CUDA graph with programmatic dependent launch and with Y1/Z/Y2 fused into one kernel per yz-plane
    // (fts_plane.cuh: two kernels per step), beat the persistent ticket kernel at 16^3 (2.55 -> 1.38 ms), 32^3 (3.25 -> 1.35 ms)
    // and 64^3 (5.19 -> 4.31 ms; one propagator 4.2 -> 2.5 ms): on these grids a step is bound by the latency of its
    // dependency hops, and a graph edge costs less than a completion counter polled through L2.
    if (c->opt.march == FTS_MARCH_AUTO && c->opt.graph && c->opt.plane && (Nx == 16 || Nx == 32 || Nx == 64)) c->persistent = 0;
    // slab size (optional): F and H of the slabs in flight must sit in L2 next to the streaming traffic
    const size_t plane = (size_t)Ny * Nz * c->esz;
    size_t target = ~(size_t)0;        // default: one slab.  Slabs cut HBM traffic from 17 to 13 E*M, but the march is not HBM-bound and
                                       // coarser phases measure 1.5-3 % faster; fts_set_option("slab_bytes") re-enables them
    if (c->opt.slab_bytes > 0) target = (size_t)c->opt.slab_bytes;
    int planes = Nx;
    while (planes > 1 && (size_t)planes * plane > target) planes >>= 1;
    while (Nx / planes > MARCH_MAXCHUNKS) planes <<= 1;
    if (c->nprop == 1 && planes == Nx && c->opt.slab_bytes <= 0) planes = Nx / 2;      // one propagator: two slabs pipeline Y1/Z/Y2 against each other (-10 % at 64^3)
    if (!c->persistent) planes = Nx;
    c->planes = planes; c->nchunks = Nx / planes;
    c->lag = c->opt.lag >= 0 ? c->opt.lag : 1;
    std::vector<Phase> all(5 * MARCH_MAXPH, mkphase(0, 0, 0, 0, 0));
    if (c->persistent) {
        phase_counts(c, mi[0], mi[1], mi[2], tz, planes, c->cnt);
        const bool inter = c->opt.interleave != 0;
        std::vector<Phase> t = make_template(c->nprop, c->nchunks, c->lag, inter, c->cnt, &c->tickets_per_round);
        if ((int)t.size() > MARCH_MAXPH) { c->err = "march template too long"; return FTS_EINVAL; }
        c->nph = (int)t.size();
        std::copy(t.begin(), t.end(), all.begin());
    }
    // per-launch templates (stream-ordered mode): kind k at all[MARCH_MAXPH*(1+k)], one phase per propagator
    int cl[4]; phase_counts(c, mi[0], mi[1], mi[2], tz, Nx, cl);
    for (int k = 0; k < 4; ++k)
        for (int b = 0; b < c->nprop; ++b) {
            all[MARCH_MAXPH * (1 + k) + b] = mkphase(b * cl[k], k, b, 0, 0);
            all[MARCH_MAXPH * (1 + k) + 2 + b] = mkphase(0, k, b, 0, 0);       // propagator b alone (see march_t)
        }
    if (!c->persistent) for (int k = 0; k < 4; ++k) c->cnt[k] = cl[k];
    CK(cudaMemcpy(c->phases, all.data(), all.size() * sizeof(Phase), cudaMemcpyHostToDevice));
    return FTS_OK;
}


// ------------------------------------------------------------------------------------------------
// TMA march (fts_march2.cuh): cubic grids with pencil length 128 or 256.  Tensor maps are encoded once per
// context through the driver entry point (no link-time dependency on libcuda).
// ------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr; cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess) fn = (EncodeTiledFn)p;
    }
    return fn;
}
static bool v2_shape_ok(const Ctx* c) { return c->g[0] == c->g[1] && c->g[1] == c->g[2] && (c->g[0] == 128 || c->g[0] == 256); }

// one field (or a store of `nslices` fields) seen as [slice][ix][iy][2 Nz scalars]; box = a strided tile along x or along y
static bool make_tile_map(const Ctx* c, CUtensorMap* m, void* base, int nslices, bool along_x) {
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return false;
    const cuuint64_t N = (cuuint64_t)c->g[0], es = c->esz;
    const cuuint64_t dims[4] = {2 * N, N, N, (cuuint64_t)nslices};
    const cuuint64_t strides[3] = {N * es, N * N * es, N * N * N * es};
    const cuuint32_t box[4] = {16, along_x ? 1u : (cuuint32_t)N, along_x ? (cuuint32_t)N : 1u, 1};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    const bool f64 = c->prec == FTS_F64;
    return enc(m, f64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               f64 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B, f64 ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B : CU_TENSOR_MAP_L2_PROMOTION_L2_64B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <class T, int N>
static cudaError_t launch_march2_inst(const Ctx* c, const March2Args& A, int grid, int* occ, cudaStream_t st) {
    typedef M2Cfg<T, N> Cfg;
    cudaError_t e = cudaFuncSetAttribute(march2_kernel<T, N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM);
    if (e != cudaSuccess) return e;
    if (occ) return cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ, march2_kernel<T, N>, M2_LAUNCH, Cfg::SMEM);
    march2_kernel<T, N><<<grid, M2_LAUNCH, Cfg::SMEM, st>>>(c->maps, A);
    g_launches += 1;
    return cudaGetLastError();
}
template <class T>
static cudaError_t launch_march2(const Ctx* c, const March2Args& A, int grid, int* occ, cudaStream_t st) {
    return c->g[0] == 256 ? launch_march2_inst<T, 256>(c, A, grid, occ, st) : launch_march2_inst<T, 128>(c, A, grid, occ, st);
}
template <class T>
static long long march2_total(const Ctx* c, int nsteps) {
    return c->g[0] == 256 ? M2Sched<T, 256>(c->nprop, c->v2_lag, c->v2_skew, nsteps).total() : M2Sched<T, 128>(c->nprop, c->v2_lag, c->v2_skew, nsteps).total();
}

template <class T>
static fts_status plan_march2(Ctx* c) {
    c->v2 = 0;
    if (!v2_shape_ok(c) || c->opt.march == FTS_MARCH_LAUNCH || c->opt.march == FTS_MARCH_TICKET) return FTS_OK;
    bool ok = true;
    for (int b = 0; b < 2 && ok; ++b) {
        const int pb = b < c->nprop ? b : 0;
        ok = ok && make_tile_map(c, &c->maps.x[M2_MAP_F + b], c->F[pb], 1, true) && make_tile_map(c, &c->maps.x[M2_MAP_H + b], c->H[pb], 1, true) &&
             make_tile_map(c, &c->maps.x[M2_MAP_E + b], (void*)e4_field(c, b), 1, true) && make_tile_map(c, &c->maps.x[M2_MAP_E + 2 + b], (void*)e4_field(c, 2 + b), 1, true) &&
             make_tile_map(c, &c->maps.x[M2_MAP_Q + b], c->q[pb], c->nslots, true) &&
             make_tile_map(c, &c->maps.y[0 + b], c->F[pb], 1, false) && make_tile_map(c, &c->maps.y[2 + b], c->H[pb], 1, false);
    }
    if (!ok) {
        if (c->opt.march == FTS_MARCH_TMA) { c->err = "cuTensorMapEncodeTiled failed or is unavailable"; return FTS_ECUDA; }
        return FTS_OK;                                    // automatic mode: fall back to the ticket march of fts_march.cuh
    }
    const int N = c->g[0], G = N == 256 ? 1 : 2, ppi = N == 256 ? 8 : 16;
    const int per_slot = c->nprop * (2 * (N / 8 / G) + 2 * (N / ppi) + N / 8 / G);
    March2Args A; std::memset(&A, 0, sizeof A);
    CK(launch_march2<T>(c, A, 0, &c->v2_occ, 0));
    if (c->v2_occ < 1) { c->err = "TMA march kernel does not fit on an SM"; return FTS_ECUDA; }
    // A phase and the phase that consumes it must be further apart in ticket order than the tickets in flight: each CTA
    // holds up to 5 (one computing, two staged, one waiting for a buffer, one drawn ahead).  Measured on B200: the march
    // time is flat from 1.25x that distance on (lag 24-32 at 128^3, 4-6 at 256^3) and rises below it.
    const int inflight = 5 * c->v2_occ * c->sms;
    int lag = (5 * inflight / 4 + per_slot - 1) / per_slot;
    if (lag > 48) lag = 48;
    if (c->opt.lag >= 0) lag = c->opt.lag;
    c->v2_lag = lag;
    c->v2_skew = c->nprop == 2 ? (c->opt.skew >= 0 ? c->opt.skew : lag) : 0;
    c->v2 = 1;
    return FTS_OK;
}

template <class T>
static fts_status march2_t(Ctx* c, int nsteps, cudaStream_t st) {
    March2Args A; std::memset(&A, 0, sizeof A);
    for (int b = 0; b < 2; ++b) { A.F[b] = c->F[b]; A.H[b] = c->H[b]; }
    for (int i = 0; i < 4; ++i) A.e4[i] = e4_field(c, i);
    A.packed = c->packed; A.seg = c->seg;
    for (int d = 0; d < 3; ++d) { A.tab[d][0] = c->dim[d].tab[0]; A.tab[d][1] = c->dim[d].tab[1]; }
    A.tw = c->dim[0].tw2;
    A.Ns = c->Ns; A.jA = c->jA; A.nspecies = c->nspecies; A.nprop = c->nprop; A.nsteps = nsteps; A.lag = c->v2_lag; A.skew = c->v2_skew;
    for (int b = 0; b < 2; ++b) A.q[b] = c->q[b < c->nprop ? b : 0];
    A.dens = dens_args(c, nsteps);
    A.cnt = c->counters; A.ticket = (unsigned*)((char*)c->counters + c->counters_bytes - 256);
    A.err = (int*)((char*)c->counters + c->counters_bytes - 128);
    long long grid = (long long)c->v2_occ * c->sms;
    const long long total = march2_total<T>(c, nsteps);
    if (grid > total) grid = total;
    CK(launch_march2<T>(c, A, (int)grid, nullptr, st));
    return FTS_OK;
}

// Fused yz-plane kernel (fts_plane.cuh) for Ny = Nz = 16, 32 or 64: replaces the Y1, Z and Y2 launches of a step.
template <class T, int N, int EPT>
static cudaError_t launch_plane_inst(const PlaneArgs& A, int grid, cudaStream_t st) {
    typedef PlaneCfg<T, N, EPT> Cfg;
    cudaError_t e = cudaFuncSetAttribute(plane_kernel<T, N, EPT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(Cfg::NT); cfg.dynamicSmemBytes = Cfg::SMEM; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization; at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    e = cudaLaunchKernelEx(&cfg, plane_kernel<T, N, EPT>, A);
    g_launches += 1;
    return e;
}
static int plane_planes_per_cta(const Ctx* c) {           // 0: the plane kernel does not apply to this grid
    const int N = c->g[1];
    if (!c->opt.plane || c->g[2] != N || (N != 16 && N != 32 && N != 64)) return 0;
    const int pl = N == 16 ? 8 : 1;
    return c->g[0] % pl == 0 ? pl : 0;
}
template <class T>
static cudaError_t launch_plane(const Ctx* c, int step, cudaStream_t st) {
    PlaneArgs A; std::memset(&A, 0, sizeof A);
    for (int b = 0; b < 2; ++b) { A.F[b] = c->F[b]; A.H[b] = c->H[b]; }
    for (int i = 0; i < 4; ++i) A.e4[i] = e4_field(c, i);
    for (int d = 0; d < 2; ++d) { A.tab[d][0] = c->dim[1 + d].tab[0]; A.tab[d][1] = c->dim[1 + d].tab[1]; A.tw[d] = c->dim[1 + d].tw; }
    A.seg = c->seg; A.Nx = c->g[0]; A.Ns = c->Ns; A.nspecies = c->nspecies; A.nprop = c->nprop; A.packed = c->packed; A.step = step;
    const int pl = plane_planes_per_cta(c), grid = c->nprop * 2 * (c->g[0] / pl);
    if (c->g[1] == 64) return launch_plane_inst<T, 64, 8>(A, grid, st);
    return c->g[1] == 16 ? launch_plane_inst<T, 16, 16>(A, grid, st) : launch_plane_inst<T, 32, 8>(A, grid, st);
}

// Straight-line T kernel (fts_plane.cuh) for x pencils of up to 64 points: replaces march_kernel's T launch of a step.
template <class T, int N, int EPT>
static cudaError_t launch_tline_inst(const TlineArgs& A, cudaStream_t st) {
    typedef TlineCfg<T, N, EPT> Cfg;
    cudaError_t e = cudaFuncSetAttribute(tline_kernel<T, N, EPT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM);
    if (e != cudaSuccess) return e;
    const int ntile = A.plane / Cfg::TZ, items = (ntile + Cfg::GPB_S - 1) / Cfg::GPB_S;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(A.nb * items); cfg.blockDim = dim3(Cfg::LAUNCH); cfg.dynamicSmemBytes = Cfg::SMEM; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization; at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    e = cudaLaunchKernelEx(&cfg, tline_kernel<T, N, EPT>, A);
    g_launches += 1;
    return e;
}
static bool tline_ok(const Ctx* c) { const int N = c->g[0]; return c->opt.tline && (N == 1 || N == 8 || N == 16 || N == 32 || N == 64) && c->g[2] % 8 == 0; }
template <class T>
static cudaError_t launch_tline(const Ctx* c, const MarchArgs& M, int step, int b0, int nb, cudaStream_t st) {
    TlineArgs A; std::memset(&A, 0, sizeof A);
    for (int b = 0; b < 2; ++b) { A.q[b] = c->q[b]; A.F[b] = c->F[b]; A.H[b] = c->H[b]; }
    for (int i = 0; i < 4; ++i) A.e4[i] = e4_field(c, i);
    A.tab[0] = c->dim[0].tab[0]; A.tab[1] = c->dim[0].tab[1]; A.tw = c->dim[0].tw;
    A.seg = c->seg; A.M = (long long)c->M; A.plane = c->g[1] * c->g[2];
    A.Ns = c->Ns; A.nspecies = c->nspecies; A.nprop = c->nprop; A.packed = c->packed; A.step = step; A.nsteps = M.nsteps;
    A.b0 = b0; A.nb = nb; A.dens = M.dens;
    switch (c->g[0]) {
        case 1: return launch_tline_inst<T, 1, 1>(A, st);
        case 8: return launch_tline_inst<T, 8, 8>(A, st);
        case 16: return launch_tline_inst<T, 16, 16>(A, st);
        case 32: return launch_tline_inst<T, 32, 8>(A, st);
        case 64: return launch_tline_inst<T, 64, 8>(A, st);
    }
    return cudaErrorInvalidValue;
}

// Per-phase launch mode: one launch per phase kind and step (stream order replaces the completion counters).
template <class T>
static fts_status march_launches_t(Ctx* c, MarchArgs A, int nsteps, cudaStream_t st) {
    static const int dim_of[4] = {0, 1, 2, 1};
    const bool planes = plane_planes_per_cta(c) > 0;       // small yz-planes: Y1, Z, Y2 fused into one kernel per step
    const bool tline = tline_ok(c);
    for (int j = 0; j <= nsteps; ++j) {
        for (int k = 0; k < 4; ++k) {
            if (k != PH_T && j == nsteps) break;
            if (k != PH_T && planes) { CK(launch_plane<T>(c, j, st)); break; }
            A.round0 = A.round1 = j;
            if (k == PH_T && tline) {                      // straight-line T kernel; split per propagator at the middle of the chain (see below)
                if (c->nprop == 2 && A.dens.on && j == A.dens.half) { CK(launch_tline<T>(c, A, j, 0, 1, st)); CK(launch_tline<T>(c, A, j, 1, 1, st)); }
                else CK(launch_tline<T>(c, A, j, 0, c->nprop, st));
                continue;
            }
            if (k == PH_T && c->nprop == 2 && A.dens.on && j == A.dens.half) {
                // the middle of the chain: q+'s item multiplies q+_h with the slice q_h that q's item of the SAME step stores
                // (DensArgs), so the two propagators' T phases cannot share a launch here
                for (int b = 0; b < 2; ++b) {
                    A.phases = c->phases + MARCH_MAXPH * (1 + k) + 2 + b; A.nphases = 1; A.tickets_per_round = c->cnt[k];
                    CK(launch_march<T>(c, c->g[dim_of[k]], A, A.tickets_per_round, false, nullptr, nullptr, st));
                }
                continue;
            }
            A.phases = c->phases + MARCH_MAXPH * (1 + k); A.nphases = c->nprop; A.tickets_per_round = c->nprop * c->cnt[k];
            CK(launch_march<T>(c, c->g[dim_of[k]], A, A.tickets_per_round, false, nullptr, nullptr, st));
        }
    }
    return FTS_OK;
}

template <class T>
static fts_status march_t(Ctx* c, int nsteps, cudaStream_t st) {
    MarchArgs A; fill_march_args<T>(c, A, nsteps);
    CK(cudaMemsetAsync(c->counters, 0, c->counters_bytes - 128, st));          // counters and ticket; the error flag stays until fts_set_fields
    if (nsteps == c->Ns && c->keep != c->Ns)                                    // S6: the density sums the T items accumulate into
        for (int b = 0; b < c->nprop; ++b) for (int a = 0; a < c->nspecies; ++a) CK(cudaMemsetAsync(c->acc[b][a], 0, c->M * c->esz, st));
    if (c->v2) return march2_t<T>(c, nsteps, st);
    if (c->persistent) {
        A.nchunks = c->nchunks; A.planes = c->planes;
        A.phases = c->phases; A.nphases = c->nph; A.tickets_per_round = c->tickets_per_round; A.round0 = 0; A.round1 = nsteps;
        A.ntT = c->cnt[PH_T]; A.nY1 = c->cnt[PH_Y1]; A.nZ = c->cnt[PH_Z]; A.nY2 = c->cnt[PH_Y2];
        A.ticket = (unsigned*)((char*)c->counters + c->counters_bytes - 256);
        if (c->occ < 1) {                              // resident CTAs per SM of this instantiation, queried once per context
            MarchInfo mi;
            CK(launch_march<T>(c, c->g[0], A, 0, true, &mi, &c->occ, st));
            if (c->occ < 1) { c->err = "march kernel does not fit on an SM"; return FTS_ECUDA; }
        }
        const int occ = c->occ;
        long long total = (long long)(nsteps + 1) * c->tickets_per_round;
        long long grid = (long long)occ * c->sms;
        if (grid > total) grid = total;
        CK(launch_march<T>(c, c->g[0], A, (int)grid, false, nullptr, nullptr, st));
        return FTS_OK;
    }
    A.nchunks = 1; A.planes = c->g[0]; A.ticket = nullptr;
    A.ntT = c->cnt[PH_T]; A.nY1 = c->cnt[PH_Y1]; A.nZ = c->cnt[PH_Z]; A.nY2 = c->cnt[PH_Y2];
    if (!c->opt.graph) return march_launches_t<T>(c, A, nsteps, st);
    // Launch-bound inner loop (4 small kernels per contour step): captured once per (context, nsteps) on a private stream and
    // replayed as one graph on the caller's stream (the caller's stream may be the legacy default stream, which cannot capture).
    for (int i = 0; i < c->ngraphs; ++i)
        if (c->graphs[i].nsteps == nsteps) { CK(cudaGraphLaunch(c->graphs[i].exec, st)); g_launches += c->graphs[i].kernels; return FTS_OK; }
    if (!c->cap_stream) CK(cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking));
    const uint64_t l0 = g_launches;
    CK(cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal));
    fts_status rc = march_launches_t<T>(c, A, nsteps, c->cap_stream);
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaStreamEndCapture(c->cap_stream, &graph);
    if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
    if (e != cudaSuccess) { c->err = std::string("cudaStreamEndCapture: ") + cudaGetErrorString(e); return FTS_ECUDA; }
    cudaGraphExec_t exec = nullptr;
    e = cudaGraphInstantiate(&exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) { c->err = std::string("cudaGraphInstantiate: ") + cudaGetErrorString(e); return FTS_ECUDA; }
    int slot;                                                                 // two shapes are kept: the first seen (normally the full march) and the latest other
    if (c->ngraphs < 2) slot = c->ngraphs++;
    else { slot = 1; cudaGraphExecDestroy(c->graphs[1].exec); }
    c->graphs[slot].exec = exec; c->graphs[slot].nsteps = nsteps; c->graphs[slot].kernels = (long long)(g_launches - l0);
    g_launches = l0;                                                          // capturing launched nothing
    CK(cudaGraphLaunch(exec, st));
    g_launches += c->graphs[slot].kernels;
    return FTS_OK;
}

template <class T>
static fts_status propagate_t(Ctx* c, int nsteps, cudaStream_t st) {
    const size_t M = c->M; const int Ns = c->Ns;
    const double ds = 1.0 / Ns;
    int* flag = (int*)((char*)c->counters + c->counters_bytes - 128);
    if (c->packed)
        boltzmann_packed_kernel<T><<<ew_blocks(M), 256, 0, st>>>((const cplx<T>*)c->f0, (const cplx<T>*)c->f1, (cplx<T>*)e4_field(c, 0), (cplx<T>*)e4_field(c, 1),
                                                                (cplx<T>*)e4_field(c, 2), (cplx<T>*)e4_field(c, 3), (int)M, ds / 4, flag);
    else
        boltzmann_kernel<T><<<ew_blocks(M), 256, 0, st>>>((const cplx<T>*)c->f0, (const cplx<T>*)c->f1, (cplx<T>*)c->e4[0], (cplx<T>*)c->e4[1], (int)M, c->P.model, ds / 4);
    g_launches += 1;
    CK(cudaGetLastError());
    fts_status rc = march_t<T>(c, nsteps, st); if (rc) return rc;
    // S7 (Eq. 4): Q = (1/M) sum_x q_Ns(x), fixed-order tree
    // (a march that gave up on a dependency leaves its error flag set: Q then becomes NaN, so that everything downstream of it --
    // densities, field updates, operators -- is visibly invalid, and every call that returns scalars reports FTS_ECUDA)
    const cplx<T>* qlast = (const cplx<T>*)c->q[0] + (size_t)slice_slot(nsteps, c->keep) * M;
    if (c->packed) CK((reduce<T, RED_SUMRE>(c, qlast, nullptr, 0.0, 1.0 / (double)M, c->scal + S_Q, st, flag)));      // z = q + i q+: Q = mean Re z
    else CK((reduce<T, RED_SUM>(c, qlast, nullptr, 0.0, 1.0 / (double)M, c->scal + S_Q, st, flag)));
    c->marched = nsteps; c->have_prop = true; c->have_phi = false; c->ops_entry = false;
    return FTS_OK;
}

// S6, last step (Eq. 8): phi = (ds / Q) (sums of q's items + sums of q+'s items); the sums were accumulated by
// the march's T items.  Written to phiA / phiB (the context's own phi fields or the caller's).
template <class T>
static fts_status density_t(Ctx* c, void* phiA, void* phiB, cudaStream_t st) {
    if (c->keep == c->Ns) {                                // full store: one streaming pass over the slices
        const cplx<T>* q = (const cplx<T>*)c->q[0];
        const cplx<T>* qd = (const cplx<T>*)c->q[c->nprop - 1];          // one propagator / packed: q+ lives in the same store
        density_store_kernel<T><<<(unsigned)((c->M + 255) / 256), 256, 0, st>>>(q, qd, c->M, c->Ns, c->cA, c->cB, c->scal + S_Q, 1.0 / c->Ns, (cplx<T>*)phiA,
                                                                                 c->nspecies == 2 ? (cplx<T>*)phiB : nullptr, c->packed);
        g_launches += 1;
        CK(cudaGetLastError());
        return FTS_OK;
    }
    if (c->packed) {
        density_finish_packed_kernel<T><<<ew_blocks(c->M), 256, 0, st>>>((const cplx<T>*)c->acc[0][0], (int)c->M, c->scal + S_Q, 1.0 / c->Ns, (cplx<T>*)phiA, (cplx<T>*)phiB);
        g_launches += 1;
        CK(cudaGetLastError());
        return FTS_OK;
    }
    const bool two = c->nprop == 2;
    density_finish_kernel<T><<<ew_blocks(c->M), 256, 0, st>>>((const cplx<T>*)c->acc[0][0], two ? (const cplx<T>*)c->acc[1][0] : nullptr,
                                                             two ? (const cplx<T>*)c->acc[0][1] : nullptr, two ? (const cplx<T>*)c->acc[1][1] : nullptr,
                                                             (int)c->M, c->scal + S_Q, 1.0 / c->Ns, (cplx<T>*)phiA, two ? (cplx<T>*)phiB : nullptr);
    g_launches += 1;
    CK(cudaGetLastError());
    return FTS_OK;
}

// F^-1{ filt(k^2) F{g} } in place: z and y forward passes, x pass with the 3-D multiplier, y and z inverse passes
template <class T>
static fts_status filter3d_t(Ctx* c, void* g, Filt f, cudaStream_t st, const void* src = nullptr) {      // src: read the field from there (g receives the result)
    PassArgs A; std::memset(&A, 0, sizeof A);
    A.job[0] = mkjob(src ? src : g, g, OP_FWD);
    CK(launch_pass<T>(c, 2, A, 1, st));
    A.job[0] = mkjob(g, g, OP_FWD);
    CK(launch_pass<T>(c, 1, A, 1, st));
    A.job[0] = mkjob(g, g, OP_FILT); A.filt = f;
    CK(launch_pass<T>(c, 0, A, 1, st));
    A.job[0] = mkjob(g, g, OP_INV);
    CK(launch_pass<T>(c, 1, A, 1, st));
    CK(launch_pass<T>(c, 2, A, 1, st));
    return FTS_OK;
}

static fts_status read_scalars(Ctx* c, double* host, int n, cudaStream_t st) {
    int flag = 0;
    CK(cudaMemcpyAsync(host, c->scal, n * sizeof(double), cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(&flag, (char*)c->counters + c->counters_bytes - 128, sizeof(int), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (flag == 3) { c->err = "real_fields is set but the fields have imaginary parts"; return FTS_EINVAL; }
    if (flag) { c->err = "march kernel: a dependency wait timed out (results invalid)"; return FTS_ECUDA; }
    return FTS_OK;
}

template <class T>
static fts_status scft_step_t(Ctx* c, double dtp, double dtm, int seidel, double* Ho, double* ro, cudaStream_t st) {
    const int M = (int)c->M; const int nb = ew_blocks(c->M);
    fts_status rc = propagate_t<T>(c, c->Ns, st); if (rc) return rc;
    rc = density_t<T>(c, c->phi[0], c->phi[1], st); if (rc) return rc;
    CK(cudaMemcpyAsync(c->scal + S_Q0, c->scal + S_Q, 2 * sizeof(double), cudaMemcpyDeviceToDevice, st));
    CK((reduce<T, RED_DIBLOCK_H>(c, c->f0, c->f1, 1.0 / c->P.chiN, 1.0 / (double)M, c->scal + S_H, st)));
    force_plus_kernel<T><<<nb, 256, 0, st>>>((const cplx<T>*)c->phi[0], (const cplx<T>*)c->phi[1], (cplx<T>*)c->G[0], M);
    g_launches += 1;
    CK((reduce<T, RED_MAXABS>(c, c->G[0], nullptr, 0.0, 1.0, c->scal + S_RP, st)));
    Filt f; f.type = FILT_RATIONAL; f.a = dtp; f.b = 0.0; f.c = dtp;                 // dt+/(1 + dt+ g_D(k^2))   (Eq. 11, reading A-10)
    rc = filter3d_t<T>(c, c->G[0], f, st); if (rc) return rc;
    add_kernel<T><<<nb, 256, 0, st>>>((cplx<T>*)c->f0, (const cplx<T>*)c->G[0], M);
    g_launches += 1;
    if (c->packed) { real_part_kernel<T><<<nb, 256, 0, st>>>((cplx<T>*)c->f0, M); g_launches += 1; }      // the complex filter leaves rounding noise in Im
    if (seidel) {
        rc = propagate_t<T>(c, c->Ns, st); if (rc) return rc;
        rc = density_t<T>(c, c->phi[0], c->phi[1], st); if (rc) return rc;
    }
    scft_minus_kernel<T><<<nb, 256, 0, st>>>((cplx<T>*)c->f1, (const cplx<T>*)c->phi[0], (const cplx<T>*)c->phi[1], (cplx<T>*)c->G[0], M, (T)(2.0 / c->P.chiN),
                                             (T)(dtm / (1.0 + dtm * 2.0 / c->P.chiN)));
    g_launches += 1;
    CK((reduce<T, RED_MAXABS>(c, c->G[0], nullptr, 0.0, 1.0, c->scal + S_RM, st)));
    double h[12];
    rc = read_scalars(c, h, 12, st); if (rc) return rc;
    c->have_prop = false;
    const double qx = h[S_Q0], qy = h[S_Q0 + 1];
    if (!std::isfinite(qx) || !std::isfinite(qy)) return FTS_ENONFINITE;
    if (Ho) { Ho[0] = h[S_H] - 0.5 * std::log(qx * qx + qy * qy); Ho[1] = h[S_H + 1] - std::atan2(qy, qx); }     // H/(CV) = mean[...] - ln Q
    if (ro) { ro[0] = h[S_RP]; ro[1] = h[S_RM]; }
    return FTS_OK;
}

// field parts of H: Edwards sum_x Omega^2 (Eq. 2), diblock mean_x [W-^2/chiN - W+] (Eq. 3)
template <class T>
static fts_status field_sums_t(Ctx* c, cudaStream_t st) {
    if (c->P.model == FTS_MODEL_EDWARDS) CK((reduce<T, RED_SUMSQ>(c, c->f0, nullptr, 0.0, 1.0, c->scal + S_SQ, st)));
    if (c->P.model == FTS_MODEL_DIBLOCK) CK((reduce<T, RED_DIBLOCK_H>(c, c->f0, c->f1, 1.0 / c->P.chiN, 1.0 / (double)c->M, c->scal + S_H, st)));
    return FTS_OK;
}

template <class T>
static fts_status cl_step_t(Ctx* c, double dt, int scheme, uint64_t seed, uint64_t step, cudaStream_t st) {
    const int M = (int)c->M; const int nb = ew_blocks(c->M);
    fts_status rc = propagate_t<T>(c, c->Ns, st); if (rc) return rc;
    rc = density_t<T>(c, c->phi[0], c->phi[1], st); if (rc) return rc;
    // the operators of the fields this step starts from cost no further solve: keep their field sums (two small reductions);
    // fts_operators after fts_cl_step then reports H, mu (and Pi) of those fields (config 4 averages them over the run)
    rc = field_sums_t<T>(c, st); if (rc) return rc;
    const double dV = c->L[0] * c->L[1] * c->L[2] / (double)c->M;
    const double lp = c->P.lambda_plus, lm = c->P.lambda_minus, ns = c->P.noise_scale;
    if (c->P.model == FTS_MODEL_EDWARDS) {
        const double amp = ns * std::sqrt(2.0 * lp * dt / dV);
        cl_edwards_kernel<T><<<nb, 256, 0, st>>>((cplx<T>*)c->f0, (const cplx<T>*)c->phi[0], (cplx<T>*)c->G[0], M, lp * dt, c->P.B, c->P.C, amp, seed, step, scheme == 0);
        g_launches += 1;
        CK(cudaGetLastError());
        if (scheme == 1) {
            Filt f; f.type = FILT_RATIONAL; f.a = 1.0; f.b = lp * dt * c->P.B; f.c = lp * dt * c->P.C;
            rc = filter3d_t<T>(c, c->G[0], f, st); if (rc) return rc;
            add_kernel<T><<<nb, 256, 0, st>>>((cplx<T>*)c->f0, (const cplx<T>*)c->G[0], M);
            g_launches += 1;
        }
    } else {
        const double ap = ns * std::sqrt(2.0 * lp * dt / dV), am = ns * std::sqrt(2.0 * lm * dt / dV);
        const double dm = scheme == 1 ? 1.0 / (1.0 + lm * dt * 2.0 * c->P.C / c->P.chiN) : 1.0;
        cl_diblock_kernel<T><<<nb, 256, 0, st>>>((cplx<T>*)c->f0, (cplx<T>*)c->f1, (const cplx<T>*)c->phi[0], (const cplx<T>*)c->phi[1], (cplx<T>*)c->G[0], M, lp * dt * c->P.C,
                                                 lm * dt * c->P.C, 2.0 / c->P.chiN, ap, am, dm, seed, step, scheme == 0);
        g_launches += 1;
        CK(cudaGetLastError());
        if (scheme == 1) {
            Filt f; f.type = FILT_RATIONAL; f.a = 1.0; f.b = 0.0; f.c = lp * dt * c->P.C;
            rc = filter3d_t<T>(c, c->G[0], f, st); if (rc) return rc;
            add_kernel<T><<<nb, 256, 0, st>>>((cplx<T>*)c->f0, (const cplx<T>*)c->G[0], M);
            g_launches += 1;
        }
    }
    CK(cudaGetLastError());
    c->have_prop = false; c->ops_entry = true;
    return FTS_OK;
}

// S10 operators (PAPER.md:50 Eq. 2, :54 Eq. 3, :183; readings A-14, A-17)
template <class T>
static fts_status operators_t(Ctx* c, double* Ho, double* muo, double* Pio, cudaStream_t st) {
    const size_t M = c->M; const int Ns = c->Ns;
    const cplx<T>* q = (const cplx<T>*)c->q[0];
    const cplx<T>* qd = (const cplx<T>*)c->q[c->nprop - 1];
    fts_status rc;
    if (Pio && c->packed) { c->err = "Pi is not available with real_fields"; return FTS_EUNSUPPORTED; }
    if (Pio && c->keep != Ns) { c->err = "Pi needs every slice of q and q+: create the context with store_both = 1"; return FTS_ESTATE; }
    if (Pio) {                                             // K_j = (1/M) sum_x q+_{Ns-j} Laplacian(q_j)
        Filt f; f.type = FILT_NEGK2; f.a = 1.0; f.b = f.c = 0.0;
        for (int j = 0; j <= Ns; ++j) {
            rc = filter3d_t<T>(c, c->G[0], f, st, q + (size_t)j * M); if (rc) return rc;      // the first pass reads the slice in place
            CK((reduce<T, RED_PROD>(c, c->G[0], qd + (size_t)(Ns - j) * M, 0.0, 1.0 / (double)M, c->kacc + 2 * j, st)));
        }
    }
    if (!c->ops_entry) { rc = field_sums_t<T>(c, st); if (rc) return rc; }      // after fts_cl_step: the sums of its entry fields are already there
    std::vector<double> kh(2 * (Ns + 1), 0.0);
    if (Pio) CK(cudaMemcpyAsync(kh.data(), c->kacc, kh.size() * sizeof(double), cudaMemcpyDeviceToHost, st));
    double h[12];
    rc = read_scalars(c, h, 12, st); if (rc) return rc;
    const double qx = h[S_Q], qy = h[S_Q + 1];
    if (!std::isfinite(qx) || !std::isfinite(qy)) return FTS_ENONFINITE;
    const double lnQ[2] = {0.5 * std::log(qx * qx + qy * qy), std::atan2(qy, qx)};
    double K[2] = {0, 0};
    if (Pio) {
        std::vector<double> wA(Ns + 1), wB(Ns + 1);
        CK(cudaMemcpy(wA.data(), c->cA, (Ns + 1) * sizeof(double), cudaMemcpyDeviceToHost));
        CK(cudaMemcpy(wB.data(), c->cB, (Ns + 1) * sizeof(double), cudaMemcpyDeviceToHost));
        double sx = 0, sy = 0;
        for (int j = 0; j <= Ns; ++j) { const double w = wA[j] + wB[j]; sx += w * kh[2 * j]; sy += w * kh[2 * j + 1]; }
        const double ds = 1.0 / Ns, den = qx * qx + qy * qy;
        K[0] = ds * (sx * qx + sy * qy) / den; K[1] = ds * (sy * qx - sx * qy) / den;
    }
    const double V = c->L[0] * c->L[1] * c->L[2], dV = V / (double)M, Cc = c->P.C, B = c->P.B;
    double H[2], mu[2], Pi[2];
    if (c->P.model == FTS_MODEL_EDWARDS) {
        H[0] = 0.5 * B * dV * h[S_SQ] - Cc * V * lnQ[0]; H[1] = 0.5 * B * dV * h[S_SQ + 1] - Cc * V * lnQ[1];
        mu[0] = std::log(Cc) - lnQ[0]; mu[1] = -lnQ[1];
        Pi[0] = Cc - 0.5 * B * dV * h[S_SQ] / V - (2.0 * Cc / 3.0) * K[0]; Pi[1] = -0.5 * B * dV * h[S_SQ + 1] / V - (2.0 * Cc / 3.0) * K[1];
    } else if (c->P.model == FTS_MODEL_DIBLOCK) {
        H[0] = h[S_H] - lnQ[0]; H[1] = h[S_H + 1] - lnQ[1];
        mu[0] = std::log(Cc > 0 ? Cc : 1.0) - lnQ[0]; mu[1] = -lnQ[1];
        Pi[0] = Cc - (2.0 * Cc / 3.0) * K[0]; Pi[1] = -(2.0 * Cc / 3.0) * K[1];
    } else {
        H[0] = -lnQ[0]; H[1] = -lnQ[1]; mu[0] = -lnQ[0]; mu[1] = -lnQ[1];
        Pi[0] = -(2.0 / 3.0) * K[0]; Pi[1] = -(2.0 / 3.0) * K[1];
    }
    if (Ho) { Ho[0] = H[0]; Ho[1] = H[1]; }
    if (muo) { muo[0] = mu[0]; muo[1] = mu[1]; }
    if (Pio) { Pio[0] = Pi[0]; Pio[1] = Pi[1]; }
    return FTS_OK;
}

static double simpson_weight(int j, int a, int b) {     // composite Simpson 1/3 on [a,b], 0 outside (reading A-5)
    if (j < a || j > b) return 0.0;
    if (j == a || j == b) return 1.0 / 3.0;
    return ((j - a) & 1) ? 4.0 / 3.0 : 2.0 / 3.0;
}

template <class T, int N, int EPT>
static void fill_tw2_shape(std::vector<cplx<T>>& tw2) {
    typedef Pencil<T, N, EPT> P; typedef PencilShape<N, EPT> S;
    if (S::ONE) return;
    for (int s = 0; s < P::TW2_SLOTS; ++s)
        for (int k1 = 0; k1 < S::R1; ++k1) {
            const long double a = 2.0L * kPiL * P::tw2_turns(s, k1);
            tw2[s * S::R1 + k1] = mk<T>((T)std::cos(a), (T)std::sin(a));
        }
}
template <class T>
static void fill_tw2(int N, std::vector<cplx<T>>& tw2) {
    switch (N) {
        case 32: fill_tw2_shape<T, 32, 8>(tw2); break;
        case 64: fill_tw2_shape<T, 64, 8>(tw2); break;
        case 128: fill_tw2_shape<T, 128, 16>(tw2); break;
        case 256: fill_tw2_shape<T, 256, 16>(tw2); break;
        default: break;
    }
}

// Chain architecture -> device tables: species per contour segment, and the Simpson weights of every slice in the density of
// species A and B (composite Simpson 1/3 per block, reading A-5: a junction slice carries 1/3 from each block it bounds).
static fts_status upload_blocks(Ctx* c) {
    const int Ns = c->Ns;
    std::vector<signed char> seg(Ns + 1, 0);
    std::vector<double> wA(Ns + 1, 0.0), wB(Ns + 1, 0.0);
    int s0 = 0;
    for (size_t i = 0; i < c->blk_steps.size(); ++i) {
        const int sp = c->blk_species[i], n = c->blk_steps[i];
        for (int j = s0; j < s0 + n; ++j) seg[j] = (signed char)sp;
        for (int j = 0; j <= Ns; ++j) (sp == 0 ? wA : wB)[j] += simpson_weight(j, s0, s0 + n);
        s0 += n;
    }
    CK(cudaMemcpy(c->seg, seg.data(), seg.size(), cudaMemcpyHostToDevice));
    CK(cudaMemcpy(c->cA, wA.data(), wA.size() * sizeof(double), cudaMemcpyHostToDevice));
    CK(cudaMemcpy(c->cB, wB.data(), wB.size() * sizeof(double), cudaMemcpyHostToDevice));
    return FTS_OK;
}

// S1: everything that is computed once per simulation
template <class T>
static fts_status build_tables(Ctx* c) {
    const double ds = 1.0 / c->Ns;
    for (int d = 0; d < 3; ++d) {
        const int N = c->g[d];
        std::vector<T> t0(N), t1(N); std::vector<cplx<T>> tw(N); std::vector<double> k2(N);
        for (int i = 0; i < N; ++i) {
            const int n = (i <= N / 2) ? i : i - N;
            const long double k = 2.0L * kPiL * (long double)n / (long double)c->L[d];
            k2[i] = (double)(k * k);
            t0[i] = (T)((double)std::exp(-(k * k) * (long double)ds) / (double)N);             // inverse-FFT 1/N folded in
            t1[i] = (T)((double)std::exp(-(k * k) * (long double)ds * 0.5L) / (double)N);
        }
        const int ept = ept_of(N), tpp = N / ept;              // twiddles per (register r, thread t): exp(-2 pi i t r / N)
        for (int r = 0; r < ept && tpp > 1; ++r)
            for (int t = 0; t < tpp; ++t) {
                const long double a = -2.0L * kPiL * (long double)(((long)t * r) % N) / (long double)N;
                tw[r * tpp + t] = mk<T>((T)std::cos(a), (T)std::sin(a));
            }
        CK(cudaMemcpy(c->dim[d].tab[0], t0.data(), N * sizeof(T), cudaMemcpyHostToDevice));
        CK(cudaMemcpy(c->dim[d].tab[1], t1.data(), N * sizeof(T), cudaMemcpyHostToDevice));
        CK(cudaMemcpy(c->dim[d].tw, tw.data(), N * sizeof(cplx<T>), cudaMemcpyHostToDevice));
        std::vector<cplx<T>> tw2(N, mk<T>(1, 0));              // twisted second stage of the FMA transform (fts_pencil.h, fwd2_b)
        fill_tw2<T>(N, tw2);
        CK(cudaMemcpy(c->dim[d].tw2, tw2.data(), N * sizeof(cplx<T>), cudaMemcpyHostToDevice));
        CK(cudaMemcpy(c->dim[d].k2, k2.data(), N * sizeof(double), cudaMemcpyHostToDevice));
    }
    fts_status rb = upload_blocks(c); if (rb) return rb;
    CK(cudaMemset(c->scal, 0, 64 * sizeof(double)));
    CK(cudaMemset(c->counters, 0, c->counters_bytes));
    return FTS_OK;
}

static void drop_graphs(Ctx* c) {
    for (int i = 0; i < c->ngraphs; ++i) if (c->graphs[i].exec) cudaGraphExecDestroy(c->graphs[i].exec);
    c->ngraphs = 0;
}

static fts_status replan(Ctx* c) {
    drop_graphs(c);
    fts_status rc = c->prec == FTS_F64 ? plan_march<double>(c) : plan_march<float>(c);
    if (!rc) rc = c->prec == FTS_F64 ? plan_march2<double>(c) : plan_march2<float>(c);
    return rc;
}

}  // namespace fts

using namespace fts;
struct fts_ctx : fts::Ctx {};

#define DISPATCH(expr_f64, expr_f32) (c->prec == FTS_F64 ? (expr_f64) : (expr_f32))

extern "C" {

const char* fts_version(void) { return "fts-b200 0.1 (sm_100a)"; }
const char* fts_last_error(const fts_ctx* c) { return c ? c->err.c_str() : "null context"; }

fts_status fts_workspace_bytes(const int grid[3], int Ns, const fts_params* P, fts_precision prec, size_t* bytes) {
    if (!bytes) return FTS_EINVAL;
    fts_status rc = validate(grid, nullptr, Ns, P, prec); if (rc) return rc;
    int g[3]; double L[3];
    squeeze_grid(grid, nullptr, g, L);
    *bytes = make_layout(g, Ns, P->model, prec == FTS_F64 ? 16 : 8, P->store_both).total;
    return FTS_OK;
}

fts_status fts_create(const int grid_user[3], const double cell_user[3], int Ns, const fts_params* P, fts_precision prec, void* ws, size_t ws_bytes, fts_ctx** out) {
    if (!cell_user || !out || !ws) return FTS_EINVAL;
    fts_status rc = validate(grid_user, cell_user, Ns, P, prec); if (rc) return rc;
    int grid[3]; double cell[3];
    squeeze_grid(grid_user, cell_user, grid, cell);
    const size_t esz = prec == FTS_F64 ? 16 : 8;
    const Layout Lo = make_layout(grid, Ns, P->model, esz, P->store_both);
    if (ws_bytes < Lo.total || ((uintptr_t)ws & 255)) return FTS_EWORKSPACE;
    fts_ctx* c = new (std::nothrow) fts_ctx;
    if (!c) return FTS_EINVAL;
    for (int d = 0; d < 3; ++d) { c->g[d] = grid[d]; c->L[d] = cell[d]; }
    c->Ns = Ns; c->P = *P; c->prec = prec; c->esz = esz;
    if (!(c->P.lambda_plus > 0)) c->P.lambda_plus = 1.0;
    if (!(c->P.lambda_minus > 0)) c->P.lambda_minus = 1.0;
    c->M = (size_t)grid[0] * grid[1] * grid[2];
    c->nprop = c->nspecies = (P->model == FTS_MODEL_DIBLOCK) ? 2 : 1;
    c->jA = (P->model == FTS_MODEL_DIBLOCK) ? (int)std::lround(P->fA * Ns) : Ns;
    if (P->model == FTS_MODEL_DIBLOCK) { c->blk_species = {0, 1}; c->blk_steps = {c->jA, Ns - c->jA}; } else { c->blk_species = {0}; c->blk_steps = {Ns}; }
    c->ws = (char*)ws; c->ws_bytes = ws_bytes;
    for (int d = 0; d < 3; ++d) {
        c->dim[d].tab[0] = c->ws + Lo.off_tab[d][0]; c->dim[d].tab[1] = c->ws + Lo.off_tab[d][1];
        c->dim[d].tw = c->ws + Lo.off_tw[d]; c->dim[d].tw2 = c->ws + Lo.off_tw2[d]; c->dim[d].k2 = (double*)(c->ws + Lo.off_k2[d]);
    }
    c->cA = (double*)(c->ws + Lo.off_cA); c->cB = (double*)(c->ws + Lo.off_cB); c->seg = (signed char*)(c->ws + Lo.off_seg);
    c->scal = (double*)(c->ws + Lo.off_scal); c->kacc = (double*)(c->ws + Lo.off_kacc); c->partial = (double2*)(c->ws + Lo.off_partial);
    c->f0 = c->ws + Lo.off_f[0]; c->f1 = c->ws + Lo.off_f[1];
    for (int i = 0; i < 2; ++i) {
        c->e4[i] = c->ws + Lo.off_e4[i]; c->F[i] = c->ws + Lo.off_F[i]; c->H[i] = c->ws + Lo.off_H[i];
        c->q[i] = c->ws + Lo.off_q[i]; c->phi[i] = c->ws + Lo.off_phi[i]; c->G[i] = c->ws + Lo.off_G[i];
        for (int a = 0; a < 2; ++a) c->acc[i][a] = c->ws + Lo.off_acc[i][a];
    }
    c->phases = (Phase*)(c->ws + Lo.off_phases); c->counters = (unsigned*)(c->ws + Lo.off_counters); c->counters_bytes = Lo.counters_bytes;
    c->keep = Lo.keep; c->nslots = Lo.nslots;
    c->have_fields = c->have_prop = c->have_phi = c->ops_entry = false; c->marched = 0; c->occ = 0;
    c->opt.march = FTS_MARCH_AUTO; c->opt.slab_bytes = 0; c->opt.lag = -1; c->opt.interleave = 1; c->opt.tz = 0; c->opt.skew = -1; c->opt.real_fields = 0; c->opt.graph = 1; c->opt.plane = 1; c->opt.tline = 1;
    c->ngraphs = 0; c->cap_stream = nullptr;
    c->packed = 0;
    c->v2 = 0; c->v2_lag = c->v2_skew = c->v2_occ = 0;
    rc = DISPATCH(build_tables<double>(c), build_tables<float>(c));
    if (!rc) rc = replan(c);
    if (rc) { delete c; return rc; }
    if (cudaDeviceSynchronize() != cudaSuccess) { delete c; return FTS_ECUDA; }      // tables and templates were written on the legacy stream
    *out = c;
    return FTS_OK;
}

fts_status fts_destroy(fts_ctx* c) {
    if (c) { drop_graphs(c); if (c->cap_stream) cudaStreamDestroy(c->cap_stream); }
    delete c;
    return FTS_OK;
}

fts_status fts_set_option(fts_ctx* c, const char* key, long long value) {
    if (!c || !key) return FTS_EINVAL;
    const auto old = c->opt;
    if (!std::strcmp(key, "march")) { if (value < 0 || value > 3) return FTS_EINVAL; c->opt.march = (int)value; }
    else if (!std::strcmp(key, "slab_bytes")) { if (value < 0) return FTS_EINVAL; c->opt.slab_bytes = value; }
    else if (!std::strcmp(key, "lag")) { if (value < -1 || value > 64) return FTS_EINVAL; c->opt.lag = (int)value; }
    else if (!std::strcmp(key, "skew")) { if (value < -1 || value > 64) return FTS_EINVAL; c->opt.skew = (int)value; }
    else if (!std::strcmp(key, "interleave")) c->opt.interleave = value != 0;
    else if (!std::strcmp(key, "tz")) { if (value != 0 && value != 8 && value != 16) return FTS_EINVAL; c->opt.tz = (int)value; }
    else if (!std::strcmp(key, "tline")) { if (value != 0 && value != 1) return FTS_EINVAL; c->opt.tline = (int)value; }
    else if (!std::strcmp(key, "plane")) { if (value != 0 && value != 1) return FTS_EINVAL; c->opt.plane = (int)value; }
    else if (!std::strcmp(key, "graph")) { if (value != 0 && value != 1) return FTS_EINVAL; c->opt.graph = (int)value; }
    else if (!std::strcmp(key, "real_fields")) {
        if (value != 0 && value != 1) return FTS_EINVAL;
        if (value && c->P.model != FTS_MODEL_DIBLOCK) return FTS_EUNSUPPORTED;      // one propagator: nothing to pack
        c->opt.real_fields = (int)value;
        c->packed = (int)value;
        c->nprop = c->packed ? 1 : c->nspecies;
    }
    else return FTS_EINVAL;
    if (c->opt.march == FTS_MARCH_TMA && !v2_shape_ok(c)) { c->opt = old; return FTS_EUNSUPPORTED; }
    c->occ = 0;
    fts_status rc = replan(c);
    if (rc) return rc;
    CK(cudaDeviceSynchronize());
    c->have_prop = false;
    return FTS_OK;
}

fts_status fts_set_blocks(fts_ctx* c, int nblocks, const int* species, const int* steps) {
    if (!c || nblocks < 1 || !species || !steps) return FTS_EINVAL;
    if (c->P.model != FTS_MODEL_DIBLOCK) return FTS_EUNSUPPORTED;
    int tot = 0;
    for (int i = 0; i < nblocks; ++i) {
        if ((species[i] != 0 && species[i] != 1) || steps[i] < 2 || (steps[i] & 1)) return FTS_EINVAL;      // reading A-5: even blocks (Simpson)
        tot += steps[i];
    }
    if (tot != c->Ns) return FTS_EINVAL;
    CK(cudaDeviceSynchronize());                           // no march may be reading the tables
    c->blk_species.assign(species, species + nblocks); c->blk_steps.assign(steps, steps + nblocks);
    fts_status rc = upload_blocks(c); if (rc) return rc;
    CK(cudaDeviceSynchronize());
    c->have_prop = false;
    return FTS_OK;
}

fts_status fts_set_fields(fts_ctx* c, const void* f0, const void* f1, void* stream) {
    if (!c || !f0 || (c->P.model == FTS_MODEL_DIBLOCK && !f1)) return FTS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaMemcpyAsync(c->f0, f0, c->M * c->esz, cudaMemcpyDeviceToDevice, st));
    if (c->P.model == FTS_MODEL_DIBLOCK) CK(cudaMemcpyAsync(c->f1, f1, c->M * c->esz, cudaMemcpyDeviceToDevice, st));
    CK(cudaMemsetAsync((char*)c->counters + c->counters_bytes - 128, 0, sizeof(int), st));      // new fields: clear a previous march's error flag
    c->have_fields = true; c->have_prop = false; c->ops_entry = false;
    return FTS_OK;
}
fts_status fts_get_fields(fts_ctx* c, void* f0, void* f1, void* stream) {
    if (!c) return FTS_EINVAL;
    if (!c->have_fields) return FTS_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    if (f0) CK(cudaMemcpyAsync(f0, c->f0, c->M * c->esz, cudaMemcpyDeviceToDevice, st));
    if (f1 && c->P.model == FTS_MODEL_DIBLOCK) CK(cudaMemcpyAsync(f1, c->f1, c->M * c->esz, cudaMemcpyDeviceToDevice, st));
    return FTS_OK;
}

fts_status fts_propagate_steps(fts_ctx* c, int nsteps, void* stream) {
    if (!c || nsteps < 0 || nsteps > c->Ns) return FTS_EINVAL;
    if (!c->have_fields) return FTS_ESTATE;
    return DISPATCH(propagate_t<double>(c, nsteps, (cudaStream_t)stream), propagate_t<float>(c, nsteps, (cudaStream_t)stream));
}
fts_status fts_propagate(fts_ctx* c, void* stream) { return c ? fts_propagate_steps(c, c->Ns, stream) : FTS_EINVAL; }

fts_status fts_density_operators(fts_ctx* c, void* phiA, void* phiB, double Q_out[2], void* stream) {
    if (!c || !phiA || (c->nspecies == 2 && !phiB)) return FTS_EINVAL;
    if (!c->have_prop || c->marched != c->Ns) return FTS_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    fts_status rc = DISPATCH(density_t<double>(c, phiA, phiB, st), density_t<float>(c, phiA, phiB, st));
    if (rc) return rc;
    double h[2];
    rc = read_scalars(c, h, 2, st); if (rc) return rc;
    if (Q_out) { Q_out[0] = h[0]; Q_out[1] = h[1]; }
    if (!std::isfinite(h[0]) || !std::isfinite(h[1])) return FTS_ENONFINITE;
    return FTS_OK;
}

fts_status fts_get_slice(fts_ctx* c, int which, int j, void* out, void* stream) {
    if (!c || !out || which < 0 || which > 1 || j < 0 || j > c->Ns) return FTS_EINVAL;
    if (!c->have_prop || j > c->marched) return FTS_ESTATE;
    if (j > c->keep && j != c->marched) { c->err = "slice not retained by the meet-in-the-middle store (store_both = 0)"; return FTS_ESTATE; }
    if (c->packed) {
        const char* z = (const char*)c->q[0] + (size_t)slice_slot(j, c->keep) * c->M * c->esz;
        if (c->prec == FTS_F64) unpack_kernel<double><<<ew_blocks(c->M), 256, 0, (cudaStream_t)stream>>>((const cplx<double>*)z, (cplx<double>*)out, (int)c->M, which);
        else unpack_kernel<float><<<ew_blocks(c->M), 256, 0, (cudaStream_t)stream>>>((const cplx<float>*)z, (cplx<float>*)out, (int)c->M, which);
        g_launches += 1;
        CK(cudaGetLastError());
        return FTS_OK;
    }
    const char* base = (const char*)c->q[which == 1 ? c->nprop - 1 : 0];
    CK(cudaMemcpyAsync(out, base + (size_t)slice_slot(j, c->keep) * c->M * c->esz, c->M * c->esz, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    return FTS_OK;
}

fts_status fts_scft_step(fts_ctx* c, double dtp, double dtm, int seidel, double H[2], double resid[2], void* stream) {
    if (!c || !(dtp > 0) || !(dtm > 0)) return FTS_EINVAL;
    if (c->P.model != FTS_MODEL_DIBLOCK) return FTS_EUNSUPPORTED;
    if (!c->have_fields) return FTS_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    return DISPATCH(scft_step_t<double>(c, dtp, dtm, seidel, H, resid, st), scft_step_t<float>(c, dtp, dtm, seidel, H, resid, st));
}

fts_status fts_cl_step(fts_ctx* c, double dt, int scheme, uint64_t seed, uint64_t step, void* stream) {
    if (!c || !(dt > 0) || scheme < 0 || scheme > 1) return FTS_EINVAL;
    if (c->P.model == FTS_MODEL_EXTERNAL) return FTS_EUNSUPPORTED;
    if (!c->have_fields) return FTS_ESTATE;
    if (c->packed) { c->err = "complex Langevin fields are complex: clear the real_fields option first"; return FTS_ESTATE; }
    cudaStream_t st = (cudaStream_t)stream;
    return DISPATCH(cl_step_t<double>(c, dt, scheme, seed, step, st), cl_step_t<float>(c, dt, scheme, seed, step, st));
}

fts_status fts_operators(fts_ctx* c, double H[2], double mu[2], double Pi[2], void* stream) {
    if (!c) return FTS_EINVAL;
    if (!(c->have_prop || c->ops_entry) || c->marched != c->Ns) return FTS_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    return DISPATCH(operators_t<double>(c, H, mu, Pi, st), operators_t<float>(c, H, mu, Pi, st));
}

// 64 FMAs per thread per iteration; returns the FMA count of the launch so the caller can turn its own event timing into FLOP/s
fts_status fts_debug_fma_peak(int precision, int iters, void* scratch_dev, size_t scratch_bytes, double* fma_count, void* stream) {
    const int blocks = 148 * 8, threads = 256;
    if (!scratch_dev || iters < 1 || scratch_bytes < (size_t)blocks * threads * 8) return FTS_EINVAL;
    if (precision == FTS_F64) fma_peak_kernel<double><<<blocks, threads, 0, (cudaStream_t)stream>>>((double*)scratch_dev, iters, 0.999999, 1e-7);
    else fma_peak_kernel<float><<<blocks, threads, 0, (cudaStream_t)stream>>>((float*)scratch_dev, iters, 0.999999f, 1e-7f);
    g_launches += 1;
    if (fma_count) *fma_count = (double)blocks * threads * 64.0 * iters;
    return cudaGetLastError() == cudaSuccess ? FTS_OK : FTS_ECUDA;
}

uint64_t fts_launch_count(void) { return g_launches; }

fts_status fts_debug_normals(uint64_t seed, uint64_t step, uint32_t field_id, uint64_t site0, size_t n, double* out_dev, void* stream) {
    if (!out_dev) return FTS_EINVAL;
    if (n == 0) return FTS_OK;
    normals_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(seed, step, field_id, site0, n, out_dev);
    g_launches += 1;
    return cudaGetLastError() == cudaSuccess ? FTS_OK : FTS_ECUDA;
}

fts_status fts_debug_philox(uint64_t seed, uint64_t step, uint32_t field_id, uint64_t site0, size_t n, uint32_t* out_dev, void* stream) {
    if (!out_dev) return FTS_EINVAL;
    if (n == 0) return FTS_OK;
    philox_words_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(seed, step, field_id, site0, n, out_dev);
    g_launches += 1;
    return cudaGetLastError() == cudaSuccess ? FTS_OK : FTS_ECUDA;
}

}  // extern "C"
