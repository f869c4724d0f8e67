// fts_kernels.cuh — sm_100a kernels of the fts-b200 hot path.
//
// (The contour march itself is fts_march.cuh.)
// pass_kernel       one launch = one 1-D pass of a 3-D transform over a field: forward, inverse, or — the x pass of the
//                   field-update filters — forward, 3-D multiplier, inverse.  Used by the SCFT / Eq. 11 updates and Pi.
// boltzmann_kernel  exp(-w ds/4) per species.
// reduce_kernel     deterministic two-level sums / max (Q of Eq. 4, H of Eq. 2-3, residuals).
// density_finish    phi = (ds/Q) x the Simpson sums the march accumulated (Eq. 8); density_store: the same
//                   sums in one streaming pass over a full slice store (store_both = 1).
// update kernels    forces of PAPER.md:84, Euler-Maruyama / semi-implicit updates of Eq. 9-11, Philox noise.
#ifndef FTS_KERNELS_CUH
#define FTS_KERNELS_CUH

#include <cuda_runtime.h>
#include <stdint.h>

#include "fts_pencil.h"

namespace fts {

enum { OP_FWD = 1, OP_INV = 2, OP_FILT = 3 };
enum { FILT_RATIONAL = 0, FILT_NEGK2 = 1 };

struct Job {                  // block-uniform description of one field's trip through a pass
    const void* in;
    void* out;
    int op;
};

struct Filt { int type; double a, b, c; };   // RATIONAL: a / (1 + b + c*g_D(k^2));  NEGK2: -a*k^2

struct PassArgs {
    Job job[4];
    const void* tw;           // exp(-2 pi i m / N), m = 0..N-1
    int pstride;              // element stride along the pencil
    int outer_stride;         // strided passes: tile -> base offset = (tile / tiles_inner)*outer_stride + (tile % tiles_inner)*TZ
    int tiles_inner;
    int ntiles;               // strided: number of [N][TZ] tiles;  contiguous: number of pencils
    Filt filt;                // OP_FILT only (x pass): 3-D multiplier built from the three k_d^2 tables
    const double* k2x; const double* k2y; const double* k2z;
    int Nz;
    double invN;
};

template <class T, int N, int EPT, int TZ>
struct PassCfg {
    typedef PencilShape<N, EPT> S;
    static constexpr bool CONTIG = (TZ == 0);
    static constexpr int TARGET = 128;
    static constexpr int GROUP = CONTIG ? S::TPP : TZ * S::TPP;                 // threads that exchange among themselves
    static constexpr int GPB = (TARGET / GROUP) > 0 ? (TARGET / GROUP) : 1;     // tiles (strided) or pencils (contiguous) per CTA
    static constexpr int THREADS = GROUP * GPB;
    static constexpr int PS = CONTIG ? contig_ps<T, N, EPT>() : 1;
    static constexpr int XELEMS = S::ONE ? 0 : (CONTIG ? GPB * PS : GPB * N * TZ);   // one exchange buffer, in complex elements
    typedef typename std::conditional<CONTIG, XchgLayout<PS, S::R2 + 1, 1>, XchgLayout<1, S::R2 * (TZ ? TZ : 1), (TZ ? TZ : 1)>>::type L;
    static constexpr size_t SMEM = (size_t)N * sizeof(cplx<T>) + 2 * (size_t)XELEMS * sizeof(cplx<T>);
};

__device__ __forceinline__ double debye_dev(double x) {          // g_D(x) = 2(e^-x + x - 1)/x^2
    if (x < 1e-2) return 1.0 - x * (1.0 / 3.0) + x * x * (1.0 / 12.0) - x * x * x * (1.0 / 60.0) + x * x * x * x * (1.0 / 360.0);
    return 2.0 * (exp(-x) + x - 1.0) / (x * x);
}
__device__ __forceinline__ double filt_eval(const Filt& f, double k2) {
    return f.type == FILT_NEGK2 ? -f.a * k2 : f.a / (1.0 + f.b + f.c * debye_dev(k2));
}

template <class T, int N, int EPT, int TZ>
__global__ void __launch_bounds__(PassCfg<T, N, EPT, TZ>::THREADS) pass_kernel(const PassArgs A) {
    typedef PassCfg<T, N, EPT, TZ> Cfg;
    typedef Pencil<T, N, EPT> P;
    typedef typename Cfg::S S;
    typedef typename Cfg::L L;
    typedef cplx<T> C;
    constexpr int TPP = S::TPP;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* s_tw = reinterpret_cast<C*>(smem_raw);
    C* s_x0 = s_tw + N;
    C* s_x1 = s_x0 + Cfg::XELEMS;

    const int tid = threadIdx.x;
    for (int i = tid; i < N; i += Cfg::THREADS) s_tw[i] = static_cast<const C*>(A.tw)[i];
    __syncthreads();

    const Job J = A.job[blockIdx.y];
    int t, p, base, ps;
    bool active;
    if constexpr (Cfg::CONTIG) {
        t = tid % TPP;
        p = tid / TPP;
        const int pencil = blockIdx.x * Cfg::GPB + p;
        active = pencil < A.ntiles;
        base = pencil * N;
        ps = 1;
    } else {
        const int zz = tid % TZ, tb = tid / (TZ * TPP);
        t = (tid / TZ) % TPP;
        const int tile = blockIdx.x * Cfg::GPB + tb;
        active = tile < A.ntiles;
        base = (tile / A.tiles_inner) * A.outer_stride + (tile % A.tiles_inner) * TZ + zz;
        ps = A.pstride;
        p = zz;
        s_x0 += tb * (N * TZ);
        s_x1 += tb * (N * TZ);
    }

    const C* in = static_cast<const C*>(J.in);
    C v[EPT];
#pragma unroll
    for (int r = 0; r < EPT; ++r) v[r] = active ? in[base + (t + TPP * r) * ps] : mk<T>(0, 0);

    auto forward = [&]() {
        P::fwd_a(v, t, s_tw);
        if constexpr (!S::ONE) {
            P::template xchg_store_a<L>(v, t, s_x0, p);
            __syncthreads();
            P::template xchg_load_b<L>(v, t, s_x0, p);
        }
        P::fwd_b(v);
    };
    auto inverse = [&]() {
        P::inv_b(v);
        if constexpr (!S::ONE) {
            P::template xchg_store_b<L>(v, t, s_x1, p);
            __syncthreads();
            P::template xchg_load_a<L>(v, t, s_x1, p);
        }
        P::inv_a(v, t, s_tw);
    };

    if (J.op == OP_FWD) {
        forward();
    } else if (J.op == OP_INV) {
        const T s = (T)A.invN;
#pragma unroll
        for (int r = 0; r < EPT; ++r) v[r] = v[r] * s;
        inverse();
    } else {                  // OP_FILT: forward, 3-D multiplier, inverse (x pass of the field-update transforms)
        forward();
        const int c = base % A.pstride;               // offset inside the yz plane = iy*Nz + iz
        const double kyz = A.k2y[c / A.Nz] + A.k2z[c % A.Nz];
#pragma unroll
        for (int r = 0; r < EPT; ++r) v[r] = v[r] * (T)(filt_eval(A.filt, A.k2x[t + TPP * r] + kyz) * A.invN);
        inverse();
    }

    C* out = static_cast<C*>(J.out);
    if (active) {
#pragma unroll
        for (int r = 0; r < EPT; ++r) out[base + (t + TPP * r) * ps] = v[r];
    }
}

// ------------------------------------------------------------------------------------------------
// elementwise kernels
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ cplx<double> cexp_d(cplx<double> z) {
    double s, c;
    sincos(z.y, &s, &c);
    const double m = exp(z.x);
    return mk<double>(m * c, m * s);
}

// S2: species field from the stored fields, then e4 = exp(-w ds/4); evaluated in fp64, rounded to T.
// model 0: w = f0; 1: w = i*f0; 2: wA = f0 - f1, wB = f0 + f1.
template <class T>
__global__ void boltzmann_kernel(const cplx<T>* f0, const cplx<T>* f1, cplx<T>* e4A, cplx<T>* e4B, int M, int model, double ds4) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < M; i += gridDim.x * blockDim.x) {
        cplx<double> a = mk<double>((double)f0[i].x, (double)f0[i].y);
        if (model == 1) a = mk<double>(-a.y, a.x);
        if (model == 2) {
            cplx<double> b = mk<double>((double)f1[i].x, (double)f1[i].y);
            cplx<double> eb = cexp_d(mk<double>(-(a.x + b.x) * ds4, -(a.y + b.y) * ds4));
            e4B[i] = mk<T>((T)eb.x, (T)eb.y);
            a = a - b;
        }
        cplx<double> ea = cexp_d(mk<double>(-a.x * ds4, -a.y * ds4));
        e4A[i] = mk<T>((T)ea.x, (T)ea.y);
    }
}

// N1 real-field fast path (fts_march.cuh, cmul): packed factor fields (exp(-w_a ds/4), exp(-w_b ds/4)) for the species pairs
// (a, b) = (A,A), (A,B), (B,A), (B,B) -> out[2a + b]; w_A = W+ - W-, w_B = W+ + W- from the REAL parts of the stored fields.
// A field that is not real (|Im| > 1e-12 (1 + |Re|)) raises *flag to 3: the declaration "real_fields" was wrong.
template <class T>
__global__ void boltzmann_packed_kernel(const cplx<T>* f0, const cplx<T>* f1, cplx<T>* o0, cplx<T>* o1, cplx<T>* o2, cplx<T>* o3, int M, double ds4, int* flag) {
    bool bad = false;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < M; i += gridDim.x * blockDim.x) {
        const double p = (double)f0[i].x, m = (double)f1[i].x;
        bad = bad || fabs((double)f0[i].y) > 1e-12 * (1.0 + fabs(p)) || fabs((double)f1[i].y) > 1e-12 * (1.0 + fabs(m));
        const T ea = (T)exp(-(p - m) * ds4), eb = (T)exp(-(p + m) * ds4);
        o0[i] = mk<T>(ea, ea); o1[i] = mk<T>(ea, eb); o2[i] = mk<T>(eb, ea); o3[i] = mk<T>(eb, eb);
    }
    if (bad) atomicExch(flag, 3);
}
// slice of q (which = 0) or q+ (which = 1) out of the packed slice z = q + i q+
template <class T>
__global__ void unpack_kernel(const cplx<T>* z, cplx<T>* out, int M, int which) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < M; i += gridDim.x * blockDim.x) out[i] = mk<T>(which ? z[i].y : z[i].x, (T)0);
}
// packed sums (A, B) as (re, im) -> phi_A, phi_B = (ds / Q) sums, Q real
template <class T>
__global__ void density_finish_packed_kernel(const cplx<T>* acc, int M, const double* Qdev, double ds, cplx<T>* phiA, cplx<T>* phiB) {
    const double f = ds / Qdev[0];
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < M; i += gridDim.x * blockDim.x) {
        phiA[i] = mk<T>((T)((double)acc[i].x * f), (T)0);
        phiB[i] = mk<T>((T)((double)acc[i].y * f), (T)0);
    }
}
template <class T>
__global__ void real_part_kernel(cplx<T>* w, int M) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < M; i += gridDim.x * blockDim.x) w[i].y = (T)0;
}

// ------------------------------------------------------------------------------------------------
// deterministic reductions: fixed grid, fixed per-thread order, fixed shared-memory tree
// ------------------------------------------------------------------------------------------------
enum { RED_SUM = 0, RED_SUMSQ = 1, RED_PROD = 2, RED_DIBLOCK_H = 3, RED_MAXABS = 4, RED_SUMRE = 5 };
constexpr int RED_BLOCKS = 592, RED_THREADS = 256;     // 4 CTAs per SM on 148 SMs

template <class T, int OP>
__device__ __forceinline__ double2 red_value(const cplx<T>* a, const cplx<T>* b, int i, double p) {
    const double ax = (double)a[i].x, ay = (double)a[i].y;
    if constexpr (OP == RED_SUM) return make_double2(ax, ay);
    else if constexpr (OP == RED_SUMRE) return make_double2(ax, 0.0);
    else if constexpr (OP == RED_SUMSQ) return make_double2(ax * ax - ay * ay, 2.0 * ax * ay);
    else if constexpr (OP == RED_PROD) { const double bx = (double)b[i].x, by = (double)b[i].y; return make_double2(ax * bx - ay * by, ax * by + ay * bx); }
    else if constexpr (OP == RED_DIBLOCK_H) {           // W-^2/chiN - W+ with a = W+, b = W-, p = 1/chiN   (Eq. 3)
        const double bx = (double)b[i].x, by = (double)b[i].y;
        return make_double2((bx * bx - by * by) * p - ax, 2.0 * bx * by * p - ay);
    } else return make_double2(sqrt(ax * ax + ay * ay), 0.0);
}
template <int OP> __device__ __forceinline__ double2 red_comb(double2 u, double2 w) {
    if constexpr (OP == RED_MAXABS) return make_double2(fmax(u.x, w.x), 0.0);
    else return make_double2(u.x + w.x, u.y + w.y);
}

template <class T, int OP>
__global__ void __launch_bounds__(RED_THREADS) reduce_partial_kernel(const cplx<T>* a, const cplx<T>* b, int M, double p, double2* partial) {
    __shared__ double2 sm[RED_THREADS];
    double2 acc = make_double2(0.0, 0.0);
    for (int i = blockIdx.x * RED_THREADS + threadIdx.x; i < M; i += gridDim.x * RED_THREADS) acc = red_comb<OP>(acc, red_value<T, OP>(a, b, i, p));
    sm[threadIdx.x] = acc;
    __syncthreads();
    for (int s = RED_THREADS / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) sm[threadIdx.x] = red_comb<OP>(sm[threadIdx.x], sm[threadIdx.x + s]);
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sm[0];
}
template <int OP>
__global__ void __launch_bounds__(1024) reduce_final_kernel(const double2* partial, int n, double scale, double* out, const int* poison) {
    __shared__ double2 sm[1024];
    sm[threadIdx.x] = threadIdx.x < n ? partial[threadIdx.x] : make_double2(0.0, 0.0);
    __syncthreads();
    for (int s = 512; s > 0; s >>= 1) {
        if (threadIdx.x < s) sm[threadIdx.x] = red_comb<OP>(sm[threadIdx.x], sm[threadIdx.x + s]);
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const bool bad = poison && *poison != 0;           // the march gave up on a dependency: make the result visibly invalid
        out[0] = bad ? __longlong_as_double(0x7ff8000000000000ll) : sm[0].x * scale;
        out[1] = bad ? __longlong_as_double(0x7ff8000000000000ll) : sm[0].y * scale;
    }
}

// ------------------------------------------------------------------------------------------------
// S6 density (Eq. 8): the Simpson sums  sum_j c_j q_j q+_{Ns-j}  are accumulated inside the march by the T
// items (fts_march.cuh DensArgs: meet-in-the-middle, one sum per propagator and species); this kernel adds the two
// propagators' sums and multiplies by ds / Q.
// ------------------------------------------------------------------------------------------------
// The same sums from a FULL slice store (store_both = 1): one streaming pass over the 2 (Ns + 1) slices, fp64 accumulators.
// On a 180 GB part this is the faster layout (the march then carries no density work): HBM-bound,
// (2 (Ns + 1) + 2) E M bytes.  packed: z_j = q_j + i q+_j in one store, product Re z_j Im z_{Ns-j} (real).
template <class T>
__global__ void __launch_bounds__(256) density_store_kernel(const cplx<T>* q, const cplx<T>* qd, size_t M, int Ns, const double* cA, const double* cB,
                                                            const double* Qdev, double ds, cplx<T>* phiA, cplx<T>* phiB, int packed) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= M) return;
    double ax = 0, ay = 0, bx = 0, by = 0;
#pragma unroll 4
    for (int j = 0; j <= Ns; ++j) {
        const cplx<T> u = q[(size_t)j * M + i], w = qd[(size_t)(Ns - j) * M + i];
        double px, py;
        if (packed) { px = (double)u.x * (double)w.y; py = 0.0; }
        else { px = (double)u.x * (double)w.x - (double)u.y * (double)w.y; py = (double)u.x * (double)w.y + (double)u.y * (double)w.x; }
        const double wa = cA[j], wb = cB[j];
        ax += wa * px; ay += wa * py;
        bx += wb * px; by += wb * py;
    }
    const double qx = Qdev[0], qy = Qdev[1], den = ds / (qx * qx + qy * qy);     // multiply by ds * conj(Q)/|Q|^2
    phiA[i] = mk<T>((T)((ax * qx + ay * qy) * den), (T)((ay * qx - ax * qy) * den));
    if (phiB) phiB[i] = mk<T>((T)((bx * qx + by * qy) * den), (T)((by * qx - bx * qy) * den));
}

template <class T>
__global__ void density_finish_kernel(const cplx<T>* a0, const cplx<T>* a1, const cplx<T>* b0, const cplx<T>* b1, int M, const double* Qdev, double ds,
                                      cplx<T>* phiA, cplx<T>* phiB) {
    const double qx = Qdev[0], qy = Qdev[1], den = ds / (qx * qx + qy * qy);     // multiply by ds * conj(Q)/|Q|^2
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < M; i += gridDim.x * blockDim.x) {
        double ax = (double)a0[i].x, ay = (double)a0[i].y;
        if (a1) { ax += (double)a1[i].x; ay += (double)a1[i].y; }
        phiA[i] = mk<T>((T)((ax * qx + ay * qy) * den), (T)((ay * qx - ax * qy) * den));
        if (phiB) {
            const double bx = (double)b0[i].x + (double)b1[i].x, by = (double)b0[i].y + (double)b1[i].y;
            phiB[i] = mk<T>((T)((bx * qx + by * qy) * den), (T)((by * qx - bx * qy) * den));
        }
    }
}

// ------------------------------------------------------------------------------------------------
// S9 noise: Philox4x32-10 (Salmon et al., SC'11) + Box-Muller, one normal per (site, field, step)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t (&o)[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        const uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = h1 ^ c1 ^ k0, n2 = h0 ^ c3 ^ k1;
        c0 = n0; c1 = l1; c2 = n2; c3 = l0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    o[0] = c0; o[1] = c1; o[2] = c2; o[3] = c3;
}
__device__ __forceinline__ double normal_dev(uint64_t seed, uint64_t step, uint32_t field_id, uint64_t site) {
    uint32_t o[4];
    philox4x32_10((uint32_t)site, (uint32_t)(site >> 32), (uint32_t)step, field_id ^ ((uint32_t)(step >> 32) << 8), (uint32_t)seed, (uint32_t)(seed >> 32), o);
    const uint64_t m1 = ((uint64_t)o[0] << 21) | (o[1] >> 11), m2 = ((uint64_t)o[2] << 21) | (o[3] >> 11);
    const double u1 = (double)(m1 + 1) * 0x1p-53, u2 = (double)(m2 + 1) * 0x1p-53;
    return sqrt(-2.0 * log(u1)) * cos(2.0 * 3.14159265358979323846264338327950288 * u2);
}
// the four raw Philox words behind normal_dev, for the bit-exact comparison with the oracle (fts_debug_philox)
__global__ void philox_words_kernel(uint64_t seed, uint64_t step, uint32_t field_id, uint64_t site0, size_t n, uint32_t* out) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint64_t site = site0 + i;
    uint32_t o[4];
    philox4x32_10((uint32_t)site, (uint32_t)(site >> 32), (uint32_t)step, field_id ^ ((uint32_t)(step >> 32) << 8), (uint32_t)seed, (uint32_t)(seed >> 32), o);
    out[4 * i] = o[0]; out[4 * i + 1] = o[1]; out[4 * i + 2] = o[2]; out[4 * i + 3] = o[3];
}
__global__ void normals_kernel(uint64_t seed, uint64_t step, uint32_t field_id, uint64_t site0, size_t n, double* out) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = normal_dev(seed, step, field_id, site0 + i);
}

// ------------------------------------------------------------------------------------------------
// S8 forces and field updates (PAPER.md:84; :102 Eq. 9; :112-118 Eq. 10-11; readings A-10, A-11, A-15)
// ------------------------------------------------------------------------------------------------
template <class T>
__global__ void force_plus_kernel(const cplx<T>* phiA, const cplx<T>* phiB, cplx<T>* g, int M) {      // F+ = phiA + phiB - 1
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < M; i += gridDim.x * blockDim.x)
        g[i] = mk<T>(phiA[i].x + phiB[i].x - (T)1, phiA[i].y + phiB[i].y);
}
template <class T>
__global__ void add_kernel(cplx<T>* w, const cplx<T>* g, int M) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < M; i += gridDim.x * blockDim.x) w[i] = w[i] + g[i];
}
// F- = 2 W-/chiN + phiB - phiA (stored in g for the residual), W- -= coef * F-
template <class T>
__global__ void scft_minus_kernel(cplx<T>* wm, const cplx<T>* phiA, const cplx<T>* phiB, cplx<T>* g, int M, T two_over_chi, T coef) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < M; i += gridDim.x * blockDim.x) {
        const cplx<T> w = wm[i];
        const cplx<T> F = mk<T>(two_over_chi * w.x + phiB[i].x - phiA[i].x, two_over_chi * w.y + phiB[i].y - phiA[i].y);
        g[i] = F;
        wm[i] = mk<T>(w.x - coef * F.x, w.y - coef * F.y);
    }
}
// diblock CL numerators: np = l+ dt C (phiA+phiB-1) + i eta+,  nm = (-l- dt C (2W-/chiN + phiB - phiA) + eta-) * dm.
// direct = 1 (Euler-Maruyama, or after the filter): fields are advanced in place; direct = 0: np -> g0, nm applied to W-.
template <class T>
__global__ void cl_diblock_kernel(cplx<T>* wp, cplx<T>* wm, const cplx<T>* phiA, const cplx<T>* phiB, cplx<T>* g0, int M, double cp, double cm,
                                  double two_over_chi, double ampp, double ampm, double dm, uint64_t seed, uint64_t step, int direct) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < M; i += gridDim.x * blockDim.x) {
        const cplx<T> a = phiA[i], b = phiB[i], m = wm[i];
        const T ep = (T)(ampp * normal_dev(seed, step, 0u, (uint64_t)i)), em = (T)(ampm * normal_dev(seed, step, 1u, (uint64_t)i));
        const cplx<T> np = mk<T>((T)cp * (a.x + b.x - (T)1), (T)cp * (a.y + b.y) + ep);
        const cplx<T> Fm = mk<T>((T)two_over_chi * m.x + b.x - a.x, (T)two_over_chi * m.y + b.y - a.y);
        const cplx<T> nm = mk<T>((-(T)cm * Fm.x + em) * (T)dm, (-(T)cm * Fm.y) * (T)dm);
        if (direct) wp[i] = wp[i] + np; else g0[i] = np;
        wm[i] = m + nm;
    }
}
// Edwards: num = -l dt (B Omega + i C phi) + eta
template <class T>
__global__ void cl_edwards_kernel(cplx<T>* om, const cplx<T>* phi, cplx<T>* g0, int M, double ldt, double B, double Cc, double amp, uint64_t seed, uint64_t step, int direct) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < M; i += gridDim.x * blockDim.x) {
        const cplx<T> o = om[i], f = phi[i];
        const cplx<T> F = mk<T>((T)B * o.x - (T)Cc * f.y, (T)B * o.y + (T)Cc * f.x);
        const T eta = (T)(amp * normal_dev(seed, step, 0u, (uint64_t)i));
        const cplx<T> num = mk<T>(-(T)ldt * F.x + eta, -(T)ldt * F.y);
        if (direct) om[i] = o + num; else g0[i] = num;
    }
}

// ------------------------------------------------------------------------------------------------
// measurement aid (bench.py): register-resident FMA chains, 8 independent accumulators per thread, so that the
// roofline's ALU denominator is a number measured on this GPU at the clocks it actually sustains
// ------------------------------------------------------------------------------------------------
template <class T>
__global__ void __launch_bounds__(256) fma_peak_kernel(T* out, int iters, T a, T b) {
    T x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = (T)(threadIdx.x + i) * (T)1e-3;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int i = 0; i < 8; ++i) x[i] = fma(x[i], a, b);
        }
    }
    T s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace fts
#endif
