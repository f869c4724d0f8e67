// Host emulation of the CTA-level pencil transform of csrc/fts_pencil.h: every "thread" is a loop
// iteration, every __syncthreads() a phase boundary.  Checks, for each supported (N, EPT):
//   forward result == O(N^2) DFT in the documented spectral layout k = t + TPP*r,
//   forward -> inverse == N * identity, and the shared-memory exchange is bank-conflict-free for
//   both CTA layouts the kernels use; and the same for the twisted FMA transform of the TMA march.
// Not the oracle: this exercises product code on the CPU.
#include <cmath>
#include <complex>
#include <cstdio>
#include <cstdlib>
#include <vector>
#include "../paper_1204_5434_b200/csrc/fts_pencil.h"

using namespace fts;
#define FTS_PS(N, EPT, T) contig_ps<T, N, EPT>()
typedef std::complex<double> cd;
static int failures = 0;

template <class T, int N, int EPT, bool strided>
void run(int npencil, double tol) {
    typedef Pencil<T, N, EPT> P; typedef typename P::S S;
    const int TPP = S::TPP;
    constexpr int TZ = 128 / (2 * sizeof(T));          // 128-byte rows: 8 complex128 or 16 complex64
    constexpr int PS_contig = contig_ps<T, N, EPT>();
    typedef typename std::conditional<strided, XchgLayout<1, S::R2 * TZ, TZ>, XchgLayout<PS_contig, S::R2 + 1, 1>>::type L;
    size_t smn = strided ? (size_t)N * TZ : (size_t)npencil * PS_contig + N + 64;
    std::vector<cplx<T>> sm(smn + 1024), tw(N);       // tw: per-(register, thread) layout of fts_pencil.h
    std::vector<cplx<double>> twd(N);
    for (int m = 0; m < N; ++m) { double a = -2 * M_PI * m / N; twd[m] = mk<double>(cos(a), sin(a)); }
    for (int r = 0; r < EPT; ++r) for (int t = 0; t < TPP; ++t) {
        const int g = r % S::G1, k1 = r / S::G1;
        double a = -2 * M_PI * (((long)(t + TPP * g) * k1) % N) / N;
        tw[r * TPP + t] = mk<T>((T)cos(a), (T)sin(a));
    }
    std::vector<std::vector<cd>> x(npencil, std::vector<cd>(N));
    srand(N * 131 + EPT);
    for (auto& p : x) for (auto& e : p) e = cd(rand() / (double)RAND_MAX - 0.5, rand() / (double)RAND_MAX - 0.5);
    // registers of every emulated thread
    std::vector<cplx<T>> regs((size_t)npencil * TPP * EPT);
    auto R = [&](int p, int t) -> cplx<T>(&)[EPT] { return *reinterpret_cast<cplx<T>(*)[EPT]>(&regs[((size_t)p * TPP + t) * EPT]); };
    for (int p = 0; p < npencil; ++p) for (int t = 0; t < TPP; ++t) for (int r = 0; r < EPT; ++r)
        R(p, t)[r] = mk<T>((T)x[p][t + TPP * r].real(), (T)x[p][t + TPP * r].imag());
    for (int p = 0; p < npencil; ++p) for (int t = 0; t < TPP; ++t) { P::fwd_a(R(p, t), t, tw.data()); P::template xchg_store_a<L>(R(p, t), t, sm.data(), p); }
    for (int p = 0; p < npencil; ++p) for (int t = 0; t < TPP; ++t) { P::template xchg_load_b<L>(R(p, t), t, sm.data(), p); P::fwd_b(R(p, t)); }
    double err = 0;
    for (int p = 0; p < npencil; ++p)
        for (int k = 0; k < N; ++k) {
            cd ref(0, 0);
            for (int n = 0; n < N; ++n) ref += x[p][n] * cd(twd[(long)k * n % N].x, twd[(long)k * n % N].y);
            cplx<T> got = R(p, k % TPP)[k / TPP];
            err = std::max(err, std::abs(ref - cd(got.x, got.y)));
        }
    for (int p = 0; p < npencil; ++p) for (int t = 0; t < TPP; ++t) { P::inv_b(R(p, t)); P::template xchg_store_b<L>(R(p, t), t, sm.data(), p); }
    for (int p = 0; p < npencil; ++p) for (int t = 0; t < TPP; ++t) { P::template xchg_load_a<L>(R(p, t), t, sm.data(), p); P::inv_a(R(p, t), t, tw.data()); }
    double err2 = 0;
    for (int p = 0; p < npencil; ++p) for (int n = 0; n < N; ++n) {
        cplx<T> got = R(p, n % TPP)[n / TPP];
        err2 = std::max(err2, std::abs(x[p][n] * (double)N - cd(got.x, got.y)));
    }
    // bank conflicts: lanes of one warp, lane = (strided ? p + TZ*t : t + TPP*p); element size decides the phase width
    int worst = 1;
    if (!S::ONE) {
        const int esz = 2 * sizeof(T), lanes_per_phase = 128 / esz, words = esz / 4;
        for (int pass = 0; pass < 2; ++pass)            // 0: A-side addressing (store_a/load_a), 1: B-side (load_b/store_b)
            for (int r = 0; r < EPT; ++r)
                for (int w0 = 0; w0 < npencil * TPP; w0 += lanes_per_phase) {
                    int hits[32] = {0};
                    for (int l = w0; l < w0 + lanes_per_phase && l < npencil * TPP; ++l) {
                        int p = strided ? l % TZ : l / TPP, t = strided ? l / TZ : l % TPP;
                        long idx;
                        if (pass == 0) { int g = r % S::G1, k1 = r / S::G1; idx = (long)p * L::PS + k1 * L::ROW + (t + TPP * g) * L::ES; }
                        else { int g2 = r % S::G2, n2 = r / S::G2; idx = (long)p * L::PS + (t + TPP * g2) * L::ROW + n2 * L::ES; }
                        hits[(idx * words) % 32]++;
                    }
                    for (int b = 0; b < 32; ++b) worst = std::max(worst, hits[b]);
                }
    }
    bool ok = err < tol * N && err2 < tol * N * N && worst == 1;
    printf("%s N=%3d EPT=%2d TPP=%2d %s fwd_err=%.2e rt_err=%.2e conflict_degree=%d %s\n", sizeof(T) == 8 ? "f64" : "f32", N, EPT, TPP,
           strided ? "strided" : "contig ", err, err2, worst, ok ? "OK" : "FAIL");
    if (!ok) ++failures;
}

// The twisted FMA transform of the TMA march (fwd2_a, exchange A -> B, fwd2_b with the two-slot twiddle table): forward result
// == O(N^2) DFT in the same spectral layout; conj o forward o conj == N * inverse.
template <class T, int N, int EPT>
void run_twisted(double tol) {
    typedef Pencil<T, N, EPT> P; typedef typename P::S S;
    const int TPP = S::TPP;
    const long double PI = 3.14159265358979323846264338327950288L;
    std::vector<cplx<T>> tw2(2 * N + 2, mk<T>(1, 0));
    for (int s = 0; s < P::TW2_SLOTS; ++s) for (int k1 = 0; k1 < S::R1; ++k1) { const long double a = 2 * PI * P::tw2_turns(s, k1); tw2[s * S::R1 + k1] = mk<T>((T)cosl(a), (T)sinl(a)); }
    std::vector<cd> x(N);
    srand(N * 7 + EPT);
    for (auto& e : x) e = cd(rand() / (double)RAND_MAX - 0.5, rand() / (double)RAND_MAX - 0.5);
    std::vector<cplx<T>> v((size_t)TPP * EPT), u((size_t)TPP * EPT);
    auto fwd = [&]() {
        for (int t = 0; t < TPP; ++t) P::fwd2_a(*reinterpret_cast<cplx<T>(*)[EPT]>(&v[(size_t)t * EPT]));
        if (S::ONE) { u = v; return; }
        for (int t = 0; t < TPP; ++t) for (int r = 0; r < EPT; ++r) { const int g2 = r % S::G2, n2 = r / S::G2; u[(size_t)t * EPT + r] = v[(size_t)n2 * EPT + t + TPP * g2]; }
        for (int t = 0; t < TPP; ++t) P::fwd2_b(*reinterpret_cast<cplx<T>(*)[EPT]>(&u[(size_t)t * EPT]), t, tw2.data());
    };
    for (int t = 0; t < TPP; ++t) for (int r = 0; r < EPT; ++r) v[(size_t)t * EPT + r] = mk<T>((T)x[t + TPP * r].real(), (T)x[t + TPP * r].imag());
    fwd();
    double err = 0;
    for (int k = 0; k < N; ++k) {
        cd ref(0, 0);
        for (int n = 0; n < N; ++n) ref += x[n] * std::polar(1.0, (double)(-2 * PI * ((long)k * n % N) / N));
        err = std::max(err, std::abs(ref - cd(u[(size_t)(k % TPP) * EPT + k / TPP].x, u[(size_t)(k % TPP) * EPT + k / TPP].y)));
    }
    for (size_t i = 0; i < u.size(); ++i) v[i] = mk<T>(u[i].x, -u[i].y);      // conj o forward o conj
    fwd();
    double err2 = 0;
    for (int n = 0; n < N; ++n) err2 = std::max(err2, std::abs(x[n] * (double)N - cd(u[(size_t)(n % TPP) * EPT + n / TPP].x, -u[(size_t)(n % TPP) * EPT + n / TPP].y)));
    const bool ok = err < tol * N && err2 < tol * N * N;
    printf("%s N=%3d EPT=%2d twisted FMA transform fwd_err=%.2e rt_err=%.2e %s\n", sizeof(T) == 8 ? "f64" : "f32", N, EPT, err, err2, ok ? "OK" : "FAIL");
    if (!ok) ++failures;
}

template <class T>
void all(double tol) {
    run_twisted<T, 8, 8>(tol); run_twisted<T, 16, 16>(tol); run_twisted<T, 32, 8>(tol); run_twisted<T, 64, 8>(tol);
    run_twisted<T, 64, 16>(tol); run_twisted<T, 128, 16>(tol); run_twisted<T, 256, 16>(tol);
    constexpr int TZ = 128 / (2 * sizeof(T));
    run<T, 8, 8, true>(TZ, tol);    run<T, 8, 8, false>(32, tol);
    run<T, 16, 16, true>(TZ, tol);  run<T, 16, 16, false>(32, tol);
    run<T, 32, 8, true>(TZ, tol);   run<T, 32, 8, false>(8, tol);
    run<T, 64, 8, true>(TZ, tol);   run<T, 64, 8, false>(4, tol);
    run<T, 64, 16, true>(TZ, tol);  run<T, 64, 16, false>(8, tol);
    run<T, 128, 16, true>(TZ, tol); run<T, 128, 16, false>(4, tol);
    run<T, 256, 16, true>(TZ, tol); run<T, 256, 16, false>(2, tol);
}

int main() {
    all<double>(2e-15);
    all<float>(1e-6);
    printf("%s\n", failures ? "FAILED" : "ALL OK");
    return failures ? 1 : 0;
}
