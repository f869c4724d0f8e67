// fts_host_steps.h — host side, part 3 of 4: what is built on a propagator solve — densities (S6, last step), the 3-D
// filter passes, the SCFT and complex-Langevin field updates (S8-S9) and the operators H, mu, Pi (S10).
#ifndef FTS_HOST_STEPS_H
#define FTS_HOST_STEPS_H

namespace fts {

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

// The same filter applied to n <= 4 fields in the same five launches (pass_kernel takes one job per blockIdx.y): field i is read
// from src[i] and its result left in g[i].  Per field the arithmetic is that of filter3d_t, bit for bit.
template <class T>
static fts_status filter3d_batch_t(Ctx* c, void* const* g, const void* const* src, int n, Filt f, cudaStream_t st) {
    PassArgs A; std::memset(&A, 0, sizeof A);
    for (int i = 0; i < n; ++i) A.job[i] = mkjob(src[i], g[i], OP_FWD);
    CK(launch_pass<T>(c, 2, A, n, st));
    for (int i = 0; i < n; ++i) A.job[i] = mkjob(g[i], g[i], OP_FWD);
    CK(launch_pass<T>(c, 1, A, n, st));
    for (int i = 0; i < n; ++i) A.job[i] = mkjob(g[i], g[i], OP_FILT);
    A.filt = f;
    CK(launch_pass<T>(c, 0, A, n, st));
    for (int i = 0; i < n; ++i) A.job[i] = mkjob(g[i], g[i], OP_INV);
    CK(launch_pass<T>(c, 1, A, n, st));
    CK(launch_pass<T>(c, 2, A, n, st));
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
        // Four slices per set of filter launches (13 launches per four slices instead of 28).  Scratch: G[0], G[1] and the context's
        // own phi fields, which are temporaries of the step calls (every step recomputes them before use).
        Filt f; f.type = FILT_NEGK2; f.a = 1.0; f.b = f.c = 0.0;
        void* const out[4] = {c->G[0], c->G[1], c->phi[0], c->phi[1]};
        for (int j0 = 0; j0 <= Ns; j0 += 4) {
            const int n = Ns + 1 - j0 < 4 ? Ns + 1 - j0 : 4;
            const void* src[4] = {nullptr, nullptr, nullptr, nullptr};
            for (int i = 0; i < n; ++i) src[i] = q + (size_t)(j0 + i) * M;                   // the first pass reads the slices in place
            rc = filter3d_batch_t<T>(c, out, src, n, f, st); if (rc) return rc;
            for (int i = 0; i < n; ++i)
                CK((reduce<T, RED_PROD>(c, out[i], qd + (size_t)(Ns - j0 - i) * M, 0.0, 1.0 / (double)M, c->kacc + 2 * (j0 + i), st)));
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

}  // namespace fts

#endif
