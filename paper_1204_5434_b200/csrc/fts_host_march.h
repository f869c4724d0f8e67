// fts_host_march.h — host side, part 2 of 4: planning and issuing the contour march (S2-S7).  Three ways to run it:
// the persistent ticket kernel (fts_march.cuh), the persistent TMA kernel for cubic 128^3 / 256^3 grids (fts_march2.cuh),
// and one launch per phase (T-line + plane kernels, fts_plane.cuh) captured once per context as a CUDA graph and replayed.
// propagate_t at the end is the one entry the C ABI calls: Boltzmann factors, the march, Q.
#ifndef FTS_HOST_MARCH_H
#define FTS_HOST_MARCH_H

namespace fts {

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
    c->marched = nsteps; c->have_prop = true; c->ops_entry = false;
    return FTS_OK;
}

}  // namespace fts

#endif
