// fts_api.cu — the C ABI declared in include/fts.h (argument checks, call-order state, dispatch on precision).  The host
// logic behind it lives in four headers included below, in dependency order: fts_host_ctx.h (context, workspace layout,
// launch helpers), fts_host_march.h (planning and issuing the contour march, S2-S7), fts_host_steps.h (densities, field
// updates, operators, S6/S8-S10), fts_host_tables.h (host-built tables, S1).  No device allocation happens here: everything
// lives in the caller's workspace.  No CPU fallback: every arithmetic step of the path is a kernel in fts_kernels.cuh.
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
#include "fts_host_ctx.h"
#include "fts_host_march.h"
#include "fts_host_steps.h"
#include "fts_host_tables.h"

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
    c->have_fields = c->have_prop = c->ops_entry = false; c->marched = 0; c->occ = 0;
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
    const auto old = c->opt; const int old_packed = c->packed, old_nprop = c->nprop;
    auto restore = [&]() { c->opt = old; c->packed = old_packed; c->nprop = old_nprop; };
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
    if (c->opt.march == FTS_MARCH_TMA && !v2_shape_ok(c)) { restore(); return FTS_EUNSUPPORTED; }
    // A march enqueued earlier (possibly on a non-blocking side stream) may still be reading the phase templates, the counters
    // or a captured graph that replan() rewrites / destroys: wait for the device first, as fts_set_blocks does.
    if (cudaError_t e = cudaDeviceSynchronize()) { restore(); c->err = cudaGetErrorString(e); return FTS_ECUDA; }
    c->occ = 0;
    fts_status rc = replan(c);
    if (rc) {                                              // leave the context as it was: old options, old plan
        const std::string why = c->err;
        restore(); c->occ = 0;
        if (replan(c) == FTS_OK) cudaDeviceSynchronize();
        c->err = why;
        return rc;
    }
    CK(cudaDeviceSynchronize());
    if (!std::strcmp(key, "real_fields") && value == 0) {
        // The march's sticky status word also carries "the fields were not real" (3), set by the packed Boltzmann kernel.  That
        // condition ends with the option; a dependency time-out (1) is a different matter and stays until fts_set_fields.
        int* flag = (int*)((char*)c->counters + c->counters_bytes - 128);
        int h = 0;
        CK(cudaMemcpy(&h, flag, sizeof(int), cudaMemcpyDeviceToHost));
        if (h == 3) CK(cudaMemset(flag, 0, sizeof(int)));
    }
    c->have_prop = false; c->ops_entry = false;           // whatever fts_cl_step left behind belongs to the old plan
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
    c->have_prop = false; c->ops_entry = false;           // Q, slices and sums kept by fts_cl_step belong to the old chain architecture
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
