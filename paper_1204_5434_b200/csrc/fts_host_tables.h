// fts_host_tables.h — host side, part 4 of 4: tables built once per context on the host (S1) — Simpson weights and species
// per contour segment, diffusion factors exp(-k^2 ds), exp(-k^2 ds/2) with 1/N folded in, FFT twiddles incl. the twisted
// second stage — and (re)planning of the march after an option change.
#ifndef FTS_HOST_TABLES_H
#define FTS_HOST_TABLES_H

namespace fts {

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

#endif
