// fts_oracle.cpp — the CPU ORACLE (TEST INFRASTRUCTURE, NOT PRODUCT CODE; see fts_oracle.h).
//
// Literal, unfused, single-threaded implementation of the discretised scheme of PAPER.md
// (Delaney & Fredrickson, arXiv 1204.5434).  Every function cites the passage it follows.
// No blocking, no separability trick, no meet-in-the-middle: full-size 3-D factor arrays,
// 3-D FFT as three nested 1-D loops, every slice of q and q+ kept.
// Shares no code with paper_1204_5434_b200/csrc.
#include "fts_oracle.h"

#include <cmath>
#include <complex>
#include <cstring>
#include <map>
#include <vector>

namespace {

const double kPi = 3.14159265358979323846264338327950288;

// ---------------------------------------------------------------------------------------------
// 1-D DFT.  Forward (sign=-1): X[k] = sum_n x[n] exp(-2 pi i k n / N), unnormalised.
// Inverse (sign=+1): x[n] = (1/N) sum_k X[k] exp(+2 pi i k n / N).   (reading A-7;
// PAPER.md:127 only says "forward and reverse fast Fourier transform".)
// ---------------------------------------------------------------------------------------------
template <class T>
const std::vector<std::complex<T>>& twiddles(int n) {           // exp(-2 pi i m / n), computed in double
    static std::map<int, std::vector<std::complex<T>>> cache;
    auto it = cache.find(n);
    if (it != cache.end()) return it->second;
    std::vector<std::complex<T>> w(n);
    for (int m = 0; m < n; ++m) {
        double a = -2.0 * kPi * (double)m / (double)n;
        w[m] = std::complex<T>((T)std::cos(a), (T)std::sin(a));
    }
    return cache.emplace(n, std::move(w)).first->second;
}

template <class T>
void dft_direct(std::complex<T>* x, int n, int sign) {           // the definition, O(n^2)
    const auto& w = twiddles<T>(n);
    std::vector<std::complex<T>> y(n);
    for (int k = 0; k < n; ++k) {
        std::complex<T> acc(0, 0);
        for (int m = 0; m < n; ++m) {
            std::complex<T> t = w[(int)(((long long)k * m) % n)];
            if (sign > 0) t = std::conj(t);
            acc += x[m] * t;
        }
        y[k] = acc;
    }
    T s = (sign > 0) ? (T)1 / (T)n : (T)1;
    for (int k = 0; k < n; ++k) x[k] = y[k] * s;
}

template <class T>
void fft1d(std::complex<T>* x, int n, int sign) {                // textbook iterative radix-2 (Cooley-Tukey)
    if (n == 1) return;
    if (n & (n - 1)) { dft_direct(x, n, sign); return; }         // not a power of two: use the definition
    const auto& w = twiddles<T>(n);
    for (int i = 1, j = 0; i < n; ++i) {                         // bit-reversal permutation
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) std::swap(x[i], x[j]);
    }
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1, stride = n / len;
        for (int base = 0; base < n; base += len)
            for (int m = 0; m < half; ++m) {
                std::complex<T> t = w[m * stride];
                if (sign > 0) t = std::conj(t);
                std::complex<T> u = x[base + m], v = x[base + m + half] * t;
                x[base + m] = u + v;
                x[base + m + half] = u - v;
            }
    }
    if (sign > 0) { T s = (T)1 / (T)n; for (int i = 0; i < n; ++i) x[i] *= s; }
}

template <class T>
void fft3d(std::vector<std::complex<T>>& a, const int g[3], int sign) {   // three nested 1-D loops
    const int Nx = g[0], Ny = g[1], Nz = g[2];
    std::vector<std::complex<T>> p;
    for (int ix = 0; ix < Nx; ++ix)                              // along z (contiguous)
        for (int iy = 0; iy < Ny; ++iy) fft1d(&a[((size_t)ix * Ny + iy) * Nz], Nz, sign);
    p.resize(Ny);
    for (int ix = 0; ix < Nx; ++ix)                              // along y
        for (int iz = 0; iz < Nz; ++iz) {
            for (int iy = 0; iy < Ny; ++iy) p[iy] = a[((size_t)ix * Ny + iy) * Nz + iz];
            fft1d(p.data(), Ny, sign);
            for (int iy = 0; iy < Ny; ++iy) a[((size_t)ix * Ny + iy) * Nz + iz] = p[iy];
        }
    p.resize(Nx);
    for (int iy = 0; iy < Ny; ++iy)                              // along x
        for (int iz = 0; iz < Nz; ++iz) {
            for (int ix = 0; ix < Nx; ++ix) p[ix] = a[((size_t)ix * Ny + iy) * Nz + iz];
            fft1d(p.data(), Nx, sign);
            for (int ix = 0; ix < Nx; ++ix) a[((size_t)ix * Ny + iy) * Nz + iz] = p[ix];
        }
}

// O1 (PAPER.md:69 Eq. 5, :127, :145): k^2 on the full FFT grid, n_d = i if i <= N_d/2 else i - N_d.
std::vector<double> build_k2(const int g[3], const double L[3]) {
    std::vector<double> k2((size_t)g[0] * g[1] * g[2]);
    for (int ix = 0; ix < g[0]; ++ix)
        for (int iy = 0; iy < g[1]; ++iy)
            for (int iz = 0; iz < g[2]; ++iz) {
                int idx[3] = {ix, iy, iz};
                double s = 0;
                for (int d = 0; d < 3; ++d) {
                    int n = (idx[d] <= g[d] / 2) ? idx[d] : idx[d] - g[d];
                    double k = 2.0 * kPi * (double)n / L[d];
                    s += k * k;
                }
                k2[((size_t)ix * g[1] + iy) * g[2] + iz] = s;
            }
    return k2;
}

double debye(double x) {                                         // PAPER.md:116 "g is a Debye function"
    if (x < 1e-2) return 1.0 - x / 3.0 + x * x / 12.0 - x * x * x / 60.0 + x * x * x * x / 360.0;   // Taylor series: avoids cancellation
    return 2.0 * (std::exp(-x) + x - 1.0) / (x * x);
}

// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11) restated from the published algorithm.
void philox(const uint32_t c_in[4], const uint32_t k_in[2], uint32_t out[4]) {
    uint32_t c[4] = {c_in[0], c_in[1], c_in[2], c_in[3]}, k[2] = {k_in[0], k_in[1]};
    for (int r = 0; r < 10; ++r) {
        if (r) { k[0] += 0x9E3779B9u; k[1] += 0xBB67AE85u; }
        uint64_t p0 = (uint64_t)0xD2511F53u * c[0], p1 = (uint64_t)0xCD9E8D57u * c[2];
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c[1] ^ k[0], n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c[3] ^ k[1], n3 = (uint32_t)p0;
        c[0] = n0; c[1] = n1; c[2] = n2; c[3] = n3;
    }
    for (int i = 0; i < 4; ++i) out[i] = c[i];
}

// DESIGN.md reading A-15: key = (seed lo, seed hi); counter = (site lo, site hi, step lo, field id ^ (step hi << 8));
// words 0-1 -> u1, words 2-3 -> u2 as 53-bit uniforms in (0,1]; Box-Muller cosine branch.
double normal_draw(uint64_t seed, uint64_t step, uint32_t field_id, uint64_t site) {
    uint32_t c[4] = {(uint32_t)site, (uint32_t)(site >> 32), (uint32_t)step, field_id ^ ((uint32_t)(step >> 32) << 8)};
    uint32_t k[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)}, o[4];
    philox(c, k, o);
    uint64_t m1 = ((uint64_t)o[0] << 21) | (o[1] >> 11), m2 = ((uint64_t)o[2] << 21) | (o[3] >> 11);
    double u1 = (double)(m1 + 1) * 0x1p-53, u2 = (double)(m2 + 1) * 0x1p-53;
    return std::sqrt(-2.0 * std::log(u1)) * std::cos(2.0 * kPi * u2);
}

// composite Simpson 1/3 weights on [a,b] (b-a even), 0 outside (reading A-5; Eq. 8)
double simpson_w(int j, int a, int b) {
    if (j < a || j > b) return 0.0;
    if (j == a || j == b) return 1.0 / 3.0;
    return ((j - a) & 1) ? 4.0 / 3.0 : 2.0 / 3.0;
}

struct CtxBase {
    virtual ~CtxBase() {}
    virtual int set_fields(const void*, const void*) = 0;
    virtual int get_fields(void*, void*) = 0;
    virtual int propagate(int nsteps) = 0;
    virtual int density(void*, void*, double*) = 0;
    virtual int get_slice(int, int, void*) = 0;
    virtual int scft_step(double, double, int, double*, double*) = 0;
    virtual int cl_step(double, int, uint64_t, uint64_t) = 0;
    virtual int operators(double*, double*, double*) = 0;
    virtual int set_blocks(int, const int*, const int*) = 0;
};

template <class T>
struct Ctx : CtxBase {
    typedef std::complex<T> cx;
    int g[3]; double L[3]; int Ns; oracle_params P; size_t M; int jA; int nspecies;
    // Chain architecture (linear multiblock copolymers use the same propagator machinery): blocks listed
    // from the s = 0 end, each with a species (0 = A, 1 = B) and a number of contour steps.  Default: one block (homopolymer)
    // or the AB diblock (jA steps of A, Ns - jA of B).
    std::vector<std::pair<int, int>> blocks;
    std::vector<double> k2;
    std::vector<T> D1, Dh;                    // exp(-k^2 ds), exp(-k^2 ds/2)   (O1)
    std::vector<cx> f0, f1;                   // stored fields
    bool have_fields = false, have_prop = false; int marched = 0;
    std::vector<std::vector<cx>> q, qd;       // every slice of q and q+ (qd empty when q+ == q)
    std::vector<cx> phiA, phiB; cx Q;

    Ctx(const int grid[3], const double cell[3], int Ns_, const oracle_params& p) : Ns(Ns_), P(p) {
        for (int d = 0; d < 3; ++d) { g[d] = grid[d]; L[d] = cell[d]; }
        M = (size_t)g[0] * g[1] * g[2];
        nspecies = (P.model == 2) ? 2 : 1;
        jA = (P.model == 2) ? (int)std::lround(P.fA * Ns) : Ns;
        if (P.model == 2) blocks = {{0, jA}, {1, Ns - jA}}; else blocks = {{0, Ns}};
        k2 = build_k2(g, L);
        const double ds = 1.0 / Ns;
        D1.resize(M); Dh.resize(M);
        for (size_t i = 0; i < M; ++i) { D1[i] = (T)std::exp(-k2[i] * ds); Dh[i] = (T)std::exp(-k2[i] * ds * 0.5); }
    }

    double V() const { return L[0] * L[1] * L[2]; }

    // species of the contour segment [j, j+1]; Simpson weight of slice j in the density of species a (composite Simpson 1/3
    // applied separately per block, reading A-5: a junction slice carries 1/3 from each block it bounds)
    int seg_species(int j) const {
        int s0 = 0;
        for (auto& b : blocks) { if (j < s0 + b.second) return b.first; s0 += b.second; }
        return blocks.back().first;
    }
    double block_weight(int a, int j) const {
        double w = 0.0; int s0 = 0;
        for (auto& b : blocks) { if (b.first == a) w += simpson_w(j, s0, s0 + b.second); s0 += b.second; }
        return w;
    }
    int set_blocks(int n, const int* species, const int* steps) override {
        if (P.model != 2) return 6;
        if (n < 1 || !species || !steps) return 1;
        int tot = 0;
        for (int i = 0; i < n; ++i) { if ((species[i] != 0 && species[i] != 1) || steps[i] < 2 || (steps[i] & 1)) return 1; tot += steps[i]; }
        if (tot != Ns) return 1;
        blocks.clear();
        for (int i = 0; i < n; ++i) blocks.push_back({species[i], steps[i]});
        have_prop = false;
        return 0;
    }

    // O2: species fields from stored fields.
    std::vector<cx> species_field(int alpha) const {
        std::vector<cx> w(M);
        if (P.model == 0) for (size_t i = 0; i < M; ++i) w[i] = f0[i];
        else if (P.model == 1) for (size_t i = 0; i < M; ++i) w[i] = cx(0, 1) * f0[i];               // chain feels i*Omega
        else for (size_t i = 0; i < M; ++i) w[i] = (alpha == 0) ? f0[i] - f1[i] : f0[i] + f1[i];     // wA = W+ - W-, wB = W+ + W-
        return w;
    }

    // O4 (Eq. 12, reading A-3): q' = (4*half(half(q)) - full(q))/3.
    static void diffuse(std::vector<cx>& u, const std::vector<T>& D, const int g[3]) {   // F^-1{ D * F{u} }
        fft3d(u, g, -1);
        for (size_t i = 0; i < u.size(); ++i) u[i] *= D[i];
        fft3d(u, g, +1);
    }
    void step(const std::vector<cx>& e2, const std::vector<cx>& e4, const std::vector<cx>& qin, std::vector<cx>& qout) const {
        std::vector<cx> full(M), half(M);
        for (size_t i = 0; i < M; ++i) full[i] = e2[i] * qin[i];
        diffuse(full, D1, g);
        for (size_t i = 0; i < M; ++i) full[i] *= e2[i];
        for (size_t i = 0; i < M; ++i) half[i] = e4[i] * qin[i];
        diffuse(half, Dh, g);
        for (size_t i = 0; i < M; ++i) half[i] *= e2[i];
        diffuse(half, Dh, g);
        for (size_t i = 0; i < M; ++i) half[i] *= e4[i];
        qout.resize(M);
        for (size_t i = 0; i < M; ++i) qout[i] = ((T)4 * half[i] - full[i]) / (T)3;
    }

    int set_fields(const void* a, const void* b) override {
        if (!a || (P.model == 2 && !b)) return 1;
        f0.assign((const cx*)a, (const cx*)a + M);
        if (P.model == 2) f1.assign((const cx*)b, (const cx*)b + M);
        have_fields = true; have_prop = false;
        return 0;
    }
    int get_fields(void* a, void* b) override {
        if (!have_fields) return 2;
        if (a) std::memcpy(a, f0.data(), M * sizeof(cx));
        if (b && P.model == 2) std::memcpy(b, f1.data(), M * sizeof(cx));
        return 0;
    }

    // O3, O5, O6, O7.
    int propagate(int nsteps) override {
        if (!have_fields) return 2;
        if (nsteps < 0) nsteps = Ns;                               // -1 = the full march
        if (nsteps > Ns) return 1;
        const T ds = (T)(1.0 / Ns);
        std::vector<std::vector<cx>> e2(nspecies), e4(nspecies);
        for (int a = 0; a < nspecies; ++a) {                       // O3: exp(-w ds/2), exp(-w ds/4)
            std::vector<cx> w = species_field(a);
            e2[a].resize(M); e4[a].resize(M);
            for (size_t i = 0; i < M; ++i) { e2[a][i] = std::exp(-w[i] * (ds / (T)2)); e4[a][i] = std::exp(-w[i] * (ds / (T)4)); }
        }
        q.assign(Ns + 1, std::vector<cx>());
        q[0].assign(M, cx(1, 0));                                  // q(x,0) = 1
        for (int j = 0; j < nsteps; ++j) {                         // O5: the species of the block that segment [j, j+1] lies in
            int a = (nspecies == 2) ? seg_species(j) : 0;
            step(e2[a], e4[a], q[j], q[j + 1]);
        }
        qd.clear();
        if (nspecies == 2) {                                       // O6: q+ indexed from the far end (reading A-2)
            qd.assign(Ns + 1, std::vector<cx>());
            qd[0].assign(M, cx(1, 0));                             // q+(x, s=1) = 1
            for (int m = 0; m < nsteps; ++m) {                     // step m of q+ crosses the segment [Ns-m-1, Ns-m]
                int a = seg_species(Ns - 1 - m);
                step(e2[a], e4[a], qd[m], qd[m + 1]);
            }
        }
        cx acc(0, 0);                                              // O7 (Eq. 4): Q = (1/M) sum_x q_Ns(x)
        for (size_t i = 0; i < M; ++i) acc += q[nsteps][i];
        Q = acc / (T)M;
        marched = nsteps; have_prop = true;
        return 0;
    }

    const std::vector<cx>& qdag(int m) const { return (nspecies == 2) ? qd[m] : q[m]; }   // homopolymer: q+ == q

    // O8 (Eq. 8; readings A-2, A-5, A-8, A-9): plain bilinear product, Simpson per block.
    void compute_density() {
        const T ds = (T)(1.0 / Ns);
        phiA.assign(M, cx(0, 0)); phiB.assign(M, cx(0, 0));
        for (int j = 0; j <= Ns; ++j) {
            T cA = (T)block_weight(0, j), cB = (T)block_weight(1, j);
            const std::vector<cx>& a = q[j]; const std::vector<cx>& b = qdag(Ns - j);
            for (size_t i = 0; i < M; ++i) {
                cx p = a[i] * b[i];
                if (cA != 0) phiA[i] += cA * p;
                if (nspecies == 2 && cB != 0) phiB[i] += cB * p;
            }
        }
        for (size_t i = 0; i < M; ++i) { phiA[i] = phiA[i] * ds / Q; phiB[i] = phiB[i] * ds / Q; }
    }
    int density(void* a, void* b, double* Qo) override {
        if (!have_prop || marched != Ns) return 2;
        compute_density();
        if (a) std::memcpy(a, phiA.data(), M * sizeof(cx));
        if (b && nspecies == 2) std::memcpy(b, phiB.data(), M * sizeof(cx));
        if (Qo) { Qo[0] = Q.real(); Qo[1] = Q.imag(); }
        return 0;
    }
    int get_slice(int which, int j, void* out) override {
        if (!have_prop || j < 0 || j > marched || !out) return have_prop ? 1 : 2;
        const std::vector<cx>& s = (which == 0) ? q[j] : qdag(j);
        std::memcpy(out, s.data(), M * sizeof(cx));
        return 0;
    }

    // readings A-10, A-17.  H/(CV) = (1/M) sum_x [W-^2/chiN - W+] - ln Q   (Eq. 3).
    std::complex<double> diblock_H() const {
        std::complex<double> acc(0, 0);
        for (size_t i = 0; i < M; ++i) {
            std::complex<double> wm(f1[i].real(), f1[i].imag()), wp(f0[i].real(), f0[i].imag());
            acc += wm * wm / P.chiN - wp;
        }
        return acc / (double)M - std::log(std::complex<double>(Q.real(), Q.imag()));
    }

    // reading A-10: W+ ascends with the Debye-linearised response implicit (Eq. 11 at zero noise);
    // W- descends with only its explicit linear term 2/chiN implicit.
    int scft_step(double dtp, double dtm, int seidel, double* Ho, double* ro) override {
        if (P.model != 2) return 6;
        int rc = propagate(Ns); if (rc) return rc;
        compute_density();
        std::complex<double> H = diblock_H();
        if (Ho) { Ho[0] = H.real(); Ho[1] = H.imag(); }
        std::vector<cx> Fp(M);
        double rp = 0, rm = 0;
        for (size_t i = 0; i < M; ++i) { Fp[i] = phiA[i] + phiB[i] - cx(1, 0); rp = std::max(rp, (double)std::abs(Fp[i])); }
        fft3d(Fp, g, -1);
        for (size_t i = 0; i < M; ++i) Fp[i] *= (T)(dtp / (1.0 + dtp * debye(k2[i])));
        fft3d(Fp, g, +1);
        for (size_t i = 0; i < M; ++i) f0[i] += Fp[i];
        if (seidel) { rc = propagate(Ns); if (rc) return rc; compute_density(); }   // Ceniceros-Fredrickson SIS ordering
        for (size_t i = 0; i < M; ++i) {
            cx Fm = (T)(2.0 / P.chiN) * f1[i] + phiB[i] - phiA[i];                   // PAPER.md:84, second mean-field equation / C
            rm = std::max(rm, (double)std::abs(Fm));
            f1[i] -= (T)(dtm / (1.0 + dtm * 2.0 / P.chiN)) * Fm;
        }
        if (ro) { ro[0] = rp; ro[1] = rm; }
        have_prop = false;
        return 0;
    }

    // readings A-11, A-15 (PAPER.md:102 Eq. 9; :112-118 Eq. 10-11; :116 noise variance 2 lambda dt / dV).
    int cl_step(double dt, int scheme, uint64_t seed, uint64_t stepno) override {
        if (P.model == 0) return 6;
        int rc = propagate(Ns); if (rc) return rc;
        compute_density();
        const double dV = V() / (double)M;
        if (P.model == 1) {                                        // Edwards: Omega' = Omega - l dt (B Omega + i C phi) + eta
            const double lam = P.lambda_plus, amp = P.noise_scale * std::sqrt(2.0 * lam * dt / dV);
            std::vector<cx> num(M);
            for (size_t i = 0; i < M; ++i) {
                cx F = (T)P.B * f0[i] + cx(0, 1) * (T)P.C * phiA[i];
                T eta = (T)(amp * normal_draw(seed, stepno, 0, i));
                num[i] = -(T)(lam * dt) * F + cx(eta, 0);
            }
            if (scheme == 1) {
                fft3d(num, g, -1);
                for (size_t i = 0; i < M; ++i) num[i] *= (T)(1.0 / (1.0 + lam * dt * (P.B + P.C * debye(k2[i]))));
                fft3d(num, g, +1);
            }
            for (size_t i = 0; i < M; ++i) f0[i] += num[i];
        } else {                                                   // diblock
            const double lp = P.lambda_plus, lm = P.lambda_minus;
            const double ap = P.noise_scale * std::sqrt(2.0 * lp * dt / dV), am = P.noise_scale * std::sqrt(2.0 * lm * dt / dV);
            std::vector<cx> np(M), nm(M);
            for (size_t i = 0; i < M; ++i) {
                cx Fp = phiA[i] + phiB[i] - cx(1, 0);
                cx Fm = (T)(2.0 / P.chiN) * f1[i] + phiB[i] - phiA[i];
                T ep = (T)(ap * normal_draw(seed, stepno, 0, i)), em = (T)(am * normal_draw(seed, stepno, 1, i));
                np[i] = (T)(lp * dt * P.C) * Fp + cx(0, ep);       // W+ = i omega+  =>  noise enters as i*eta
                nm[i] = -(T)(lm * dt * P.C) * Fm + cx(em, 0);
            }
            if (scheme == 1) {
                fft3d(np, g, -1);
                for (size_t i = 0; i < M; ++i) np[i] *= (T)(1.0 / (1.0 + lp * dt * P.C * debye(k2[i])));
                fft3d(np, g, +1);
                const T dm = (T)(1.0 / (1.0 + lm * dt * 2.0 * P.C / P.chiN));
                for (size_t i = 0; i < M; ++i) nm[i] *= dm;
            }
            for (size_t i = 0; i < M; ++i) { f0[i] += np[i]; f1[i] += nm[i]; }
        }
        have_prop = false;
        return 0;
    }

    // readings A-14, A-17 (PAPER.md:50 Eq. 2, :54 Eq. 3, :183).  Needs a completed propagate().
    int operators(double* Ho, double* muo, double* Pio) override {
        if (!have_prop || marched != Ns) return 2;
        typedef std::complex<double> cd;
        const cd Qd(Q.real(), Q.imag()), lnQ = std::log(Qd);
        const T ds = (T)(1.0 / Ns);
        // K = (ds/Q) sum_j c_j (1/M) sum_x q+_{Ns-j} F^-1{ -k^2 F{q_j} }
        cd K(0, 0);
        for (int j = 0; j <= Ns; ++j) {
            double c = block_weight(0, j) + ((nspecies == 2) ? block_weight(1, j) : 0.0);
            std::vector<cx> lap = q[j];
            fft3d(lap, g, -1);
            for (size_t i = 0; i < M; ++i) lap[i] *= (T)(-k2[i]);
            fft3d(lap, g, +1);
            const std::vector<cx>& b = qdag(Ns - j);
            cd s(0, 0);
            for (size_t i = 0; i < M; ++i) { cx p = b[i] * lap[i]; s += cd(p.real(), p.imag()); }
            K += c * s / (double)M;
        }
        K = K * (double)ds / Qd;
        cd H(0, 0), mu(0, 0), Pi(0, 0);
        if (P.model == 1) {
            cd s2(0, 0);
            for (size_t i = 0; i < M; ++i) { cd o(f0[i].real(), f0[i].imag()); s2 += o * o; }
            const double dV = V() / (double)M;
            H = 0.5 * P.B * dV * s2 - P.C * V() * lnQ;
            mu = std::log(P.C) - lnQ;
            Pi = P.C - 0.5 * P.B * dV * s2 / V() - (2.0 * P.C / 3.0) * K;
        } else if (P.model == 2) {
            H = diblock_H();
            mu = std::log(P.C > 0 ? P.C : 1.0) - lnQ;
            Pi = P.C - (2.0 * P.C / 3.0) * K;
        } else {
            H = -lnQ; mu = -lnQ; Pi = -(2.0 / 3.0) * K;
        }
        if (Ho) { Ho[0] = H.real(); Ho[1] = H.imag(); }
        if (muo) { muo[0] = mu.real(); muo[1] = mu.imag(); }
        if (Pio) { Pio[0] = Pi.real(); Pio[1] = Pi.imag(); }
        return 0;
    }
};

}  // namespace

struct oracle_ctx { CtxBase* impl; };

extern "C" {

int oracle_create(const int grid[3], const double cell[3], int Ns, const oracle_params* p, int precision, oracle_ctx** out) {
    if (!grid || !cell || !p || !out) return 1;
    for (int d = 0; d < 3; ++d) if (grid[d] < 1 || !(cell[d] > 0)) return 1;
    if (Ns < 2 || p->model < 0 || p->model > 2) return 1;
    if (p->model == 2) {                                           // readings A-4, A-5
        double x = p->fA * Ns; long j = std::lround(x);
        if (std::fabs(x - (double)j) > 1e-9 || j <= 0 || j >= Ns) return 1;
        if ((j & 1) || ((Ns - j) & 1)) return 1;
        if (!(p->chiN > 0)) return 1;
    } else if (Ns & 1) return 1;
    oracle_ctx* c = new oracle_ctx;
    if (precision == 0) c->impl = new Ctx<double>(grid, cell, Ns, *p);
    else if (precision == 1) c->impl = new Ctx<float>(grid, cell, Ns, *p);
    else { delete c; return 1; }
    *out = c;
    return 0;
}
void oracle_destroy(oracle_ctx* c) { if (c) { delete c->impl; delete c; } }
int oracle_set_fields(oracle_ctx* c, const void* a, const void* b) { return c ? c->impl->set_fields(a, b) : 1; }
int oracle_get_fields(oracle_ctx* c, void* a, void* b) { return c ? c->impl->get_fields(a, b) : 1; }
int oracle_propagate(oracle_ctx* c) { return c ? c->impl->propagate(-1) : 1; }
int oracle_propagate_steps(oracle_ctx* c, int n) { return c ? c->impl->propagate(n) : 1; }
int oracle_set_blocks(oracle_ctx* c, int n, const int* species, const int* steps) { return c ? c->impl->set_blocks(n, species, steps) : 1; }
int oracle_density_operators(oracle_ctx* c, void* a, void* b, double Q[2]) { return c ? c->impl->density(a, b, Q) : 1; }
int oracle_get_slice(oracle_ctx* c, int which, int j, void* out) { return c ? c->impl->get_slice(which, j, out) : 1; }
int oracle_scft_step(oracle_ctx* c, double dp, double dm, int seidel, double H[2], double r[2]) { return c ? c->impl->scft_step(dp, dm, seidel, H, r) : 1; }
int oracle_cl_step(oracle_ctx* c, double dt, int scheme, uint64_t seed, uint64_t step) { return c ? c->impl->cl_step(dt, scheme, seed, step) : 1; }
int oracle_operators(oracle_ctx* c, double H[2], double mu[2], double Pi[2]) { return c ? c->impl->operators(H, mu, Pi) : 1; }

void oracle_fft1d(double* d, int n, int sign) { fft1d(reinterpret_cast<std::complex<double>*>(d), n, sign); }
void oracle_dft1d_direct(double* d, int n, int sign) { dft_direct(reinterpret_cast<std::complex<double>*>(d), n, sign); }

int oracle_rqm4_step(const int grid[3], const double cell[3], double ds, const void* w, const void* qin, void* qout) {
    typedef std::complex<double> cd;
    oracle_params p; std::memset(&p, 0, sizeof p); p.model = 0;
    Ctx<double> c(grid, cell, 2, p);                               // tables rebuilt below for the requested ds
    for (size_t i = 0; i < c.M; ++i) { c.D1[i] = std::exp(-c.k2[i] * ds); c.Dh[i] = std::exp(-c.k2[i] * ds * 0.5); }
    std::vector<cd> e2(c.M), e4(c.M), a((const cd*)qin, (const cd*)qin + c.M), b;
    const cd* wf = (const cd*)w;
    for (size_t i = 0; i < c.M; ++i) { e2[i] = std::exp(-wf[i] * (ds / 2)); e4[i] = std::exp(-wf[i] * (ds / 4)); }
    c.step(e2, e4, a, b);
    std::memcpy(qout, b.data(), c.M * sizeof(cd));
    return 0;
}
void oracle_philox4x32_10(const uint32_t c[4], const uint32_t k[2], uint32_t out[4]) { philox(c, k, out); }
double oracle_normal(uint64_t seed, uint64_t step, uint32_t field_id, uint64_t site) { return normal_draw(seed, step, field_id, site); }
double oracle_debye(double x) { return debye(x); }

}  // extern "C"
