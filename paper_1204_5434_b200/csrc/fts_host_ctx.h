// fts_host_ctx.h — host side, part 1 of 4 (included by fts_api.cu only, in this order: ctx, march, steps, tables).
// The context, the workspace layout (the single place that decides where things live), argument validation, the CK
// error macro, and the small launch helpers every other part uses: one 1-D pass of a 3-D transform (pass_kernel) and the
// deterministic two-stage reductions.  No device allocation: everything lives in the caller's workspace.
#ifndef FTS_HOST_CTX_H
#define FTS_HOST_CTX_H

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
    bool have_fields, have_prop; int marched;
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

}  // namespace fts

#endif
