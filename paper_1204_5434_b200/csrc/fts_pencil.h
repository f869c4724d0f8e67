// fts_pencil.h — register-resident 1-D pencil transforms for the fused diffusion passes.
//
// A "pencil" is one line of N grid points along x, y or z.  TPP = N/EPT threads share a pencil, each
// holding EPT complex values in registers.  The transform of length N = R1*R2 is two register-level
// radix-R butterflies (R <= 16) with ONE shared-memory exchange between them; for N <= 16 a single
// thread holds the whole pencil and no exchange is needed.  Used as forward -> multiply by a real table
// -> inverse, which is the operator exp(ds * d^2/dx_d^2) of PAPER.md:124-127 (Eq. 12) along one dimension;
// the 3-D operator is the product of the three 1-D ones because exp(-k^2 ds) factorises.
//
// Layout facts the kernels rely on (checked on the host by tests/host_pencil_test.cpp):
//   * natural layout:  register r of thread t holds point  n = t + TPP*r
//   * spectral layout: register r of thread t holds mode   k = t + TPP*r   (same map: tables need no permutation)
//
// Everything here is __host__ __device__ so the index arithmetic can be exercised on the CPU.
#ifndef FTS_PENCIL_H
#define FTS_PENCIL_H

#if defined(__CUDACC__)
#define FTS_HD __host__ __device__ __forceinline__
#else
#define FTS_HD inline
#endif

#include <type_traits>

namespace fts {

template <class T> struct alignas(2 * sizeof(T)) cplx { T x, y; };

template <class T> FTS_HD cplx<T> mk(T a, T b) { cplx<T> r; r.x = a; r.y = b; return r; }
template <class T> FTS_HD cplx<T> operator+(cplx<T> a, cplx<T> b) { return mk<T>(a.x + b.x, a.y + b.y); }
template <class T> FTS_HD cplx<T> operator-(cplx<T> a, cplx<T> b) { return mk<T>(a.x - b.x, a.y - b.y); }
template <class T> FTS_HD cplx<T> operator*(cplx<T> a, cplx<T> b) { return mk<T>(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
template <class T> FTS_HD cplx<T> operator*(cplx<T> a, T s) { return mk<T>(a.x * s, a.y * s); }
template <class T> FTS_HD cplx<T> conj(cplx<T> a) { return mk<T>(a.x, -a.y); }

// complex64 on sm_100a: Blackwell's packed fp32 pair instructions (add/sub/mul/fma.f32x2 -> FADD2 / FMUL2 / FFMA2) do a
// complex add in ONE instruction and a complex multiply in TWO (the (-y, x) swizzle is an operand modifier), which halves
// the issue slots of the fp32 butterflies — the complex64 path is bound by instruction issue, not by the fp32 pipe.
#if defined(__CUDA_ARCH__)
__device__ __forceinline__ unsigned long long pk(float lo, float hi) { unsigned long long r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ cplx<float> unpk(unsigned long long r) { cplx<float> c; asm("mov.b64 {%0, %1}, %2;" : "=f"(c.x), "=f"(c.y) : "l"(r)); return c; }
__device__ __forceinline__ cplx<float> operator+(cplx<float> a, cplx<float> b) {
    unsigned long long r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk(a.x, a.y)), "l"(pk(b.x, b.y))); return unpk(r);
}
__device__ __forceinline__ cplx<float> operator-(cplx<float> a, cplx<float> b) {
    unsigned long long r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk(a.x, a.y)), "l"(pk(b.x, b.y))); return unpk(r);
}
__device__ __forceinline__ cplx<float> operator*(cplx<float> a, cplx<float> b) {      // (ax bx - ay by, ay bx + ax by)
    unsigned long long t, r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(t) : "l"(pk(a.x, a.y)), "l"(pk(b.x, b.x)));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(pk(-a.y, a.x)), "l"(pk(b.y, b.y)), "l"(t));
    return unpk(r);
}
__device__ __forceinline__ cplx<float> operator*(cplx<float> a, float s) {
    unsigned long long r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk(a.x, a.y)), "l"(pk(s, s))); return unpk(r);
}
#endif

// cos(2 pi m / 16), m = 0..4, correctly rounded literals; everything else by symmetry.
FTS_HD constexpr double cos16_q(int m) {
    return m == 0 ? 1.0 : m == 1 ? 0.92387953251128675613 : m == 2 ? 0.70710678118654752440 : m == 3 ? 0.38268343236508977173 : 0.0;
}
FTS_HD constexpr double cos16(int m) {          // any integer m
    m = ((m % 16) + 16) % 16;
    return m <= 4 ? cos16_q(m) : m <= 8 ? -cos16_q(8 - m) : m <= 12 ? -cos16_q(m - 8) : cos16_q(16 - m);
}
FTS_HD constexpr double sin16(int m) { return cos16(m - 4); }

// multiply by exp(DIR * 2 pi i * NUM / 16) with the trivial cases folded at compile time
template <int NUM, int DIR, class T>
FTS_HD cplx<T> mul_w16(cplx<T> a) {
    constexpr int m = (((NUM * (DIR < 0 ? -1 : 1)) % 16) + 16) % 16;
    if constexpr (m == 0) return a;
    else if constexpr (m == 4) return mk<T>(-a.y, a.x);      // * i
    else if constexpr (m == 8) return mk<T>(-a.x, -a.y);
    else if constexpr (m == 12) return mk<T>(a.y, -a.x);     // * -i
    else if constexpr (m % 4 == 2 && sizeof(T) == 4) {       // complex64: a packed complex multiply (2 instructions) is cheaper
        return a * mk<T>((T)cos16(m), (T)sin16(m));
    } else if constexpr (m % 4 == 2) {                       // (+-1 +- i)/sqrt(2): 2 adds + 2 muls
        constexpr T h = (T)0.70710678118654752440;
        constexpr T sc = (T)(cos16(m) > 0 ? 1 : -1), ss = (T)(sin16(m) > 0 ? 1 : -1);
        return mk<T>((sc * a.x - ss * a.y) * h, (ss * a.x + sc * a.y) * h);
    } else {
        return a * mk<T>((T)cos16(m), (T)sin16(m));
    }
}

template <int B, int E, class F>
FTS_HD void static_for(F&& f) {
    if constexpr (B < E) {
        f(std::integral_constant<int, B>{});
        static_for<B + 1, E>(f);
    }
}

constexpr int bitrev(int i, int bits) { int r = 0; for (int b = 0; b < bits; ++b) r |= ((i >> b) & 1) << (bits - 1 - b); return r; }
constexpr int ilog2(int n) { int l = 0; while ((1 << l) < n) ++l; return l; }

// In-register DFT of R = 2,4,8,16 points held at v[OFF + S*i], i = 0..R-1.  DIR = -1 forward (e^{-i...}),
// +1 inverse (unnormalised).  Decimation in frequency, radix-2 stages, natural order in and out
// (the bit reversal is a compile-time register renaming).
template <int R, int S, int OFF, int DIR, class T, int NV>
FTS_HD void dft_reg(cplx<T> (&v)[NV]) {
    if constexpr (R > 1) {
        static_for<0, ilog2(R)>([&](auto st) {
            constexpr int half = R >> (decltype(st)::value + 1);
            static_for<0, R / 2>([&](auto bi) {
                constexpr int b = decltype(bi)::value;
                constexpr int base = (b / half) * 2 * half, i = b % half;
                constexpr int p0 = OFF + S * (base + i), p1 = OFF + S * (base + i + half);
                cplx<T> a = v[p0], c = v[p1];
                v[p0] = a + c;
                v[p1] = mul_w16<i * (8 / half), DIR>(a - c);
            });
        });
        cplx<T> tmp[R];
        static_for<0, R>([&](auto ii) { constexpr int i = decltype(ii)::value; tmp[i] = v[OFF + S * bitrev(i, ilog2(R))]; });
        static_for<0, R>([&](auto ii) { constexpr int i = decltype(ii)::value; v[OFF + S * i] = tmp[i]; });
    }
}

// ------------------------------------------------------------------------------------------------
// "Twisted" radix-2 DIF transform with FMA butterflies (used by the TMA march, fts_march2.cuh).
//
//   X[k] = sum_n x[n] (zeta w^k)^n,  w = exp(-2 pi i / R),  n, k = 0..R-1          (zeta = 1: the plain DFT)
//
// Splitting n = n' + (R/2) b gives  u = x[n'] + zeta^(R/2) x[n'+R/2]  (even k, same zeta) and
// d = x[n'] - zeta^(R/2) x[n'+R/2]  (odd k, zeta' = zeta w), so EVERY butterfly has the form a +- W c with one W per
// block: at level L (block size Rc = R / 2^(L-1)) block number blk uses  W = zeta^(Rc/2) * exp(-2 pi i E / 2^L),
// E = bitrev(blk, L-1) < 2^(L-1).  The inter-stage twiddle of the two-stage pencil transform (zeta = exp(-2 pi i k1/N))
// is thereby folded into the second stage's butterflies: no separate complex multiplies, and per level only
// max(1, 2^(L-2)) distinct W are loaded (E >= 2^(L-2) is the same W times -i, an operand swap).
// Cost per butterfly: 4 FMA for a + W c and 2 FMA for a - W c = 2a - (a + W c)  (6 fp64 instructions instead of the
// 4 + 4 of "multiply, then add and subtract"); trivial W (1, -i) cost 4 adds; (+-1 -+ i)/sqrt2 costs 2 adds + 4 FMA.
// A 128-point transform (16 x 8) needs 18.25 fp64 instructions per point instead of 23.5, a 256-point one 21.25
// instead of 27.  Output X[k] is left at position bitrev(k) and renamed to natural order at compile time.
// ------------------------------------------------------------------------------------------------
template <class T> FTS_HD cplx<T> cmadd(cplx<T> a, cplx<T> w, cplx<T> c) {          // a + w c
    if constexpr (sizeof(T) == 8) {
#if defined(__CUDA_ARCH__)
        return mk<T>(fma(-w.y, c.y, fma(w.x, c.x, a.x)), fma(w.y, c.x, fma(w.x, c.y, a.y)));
#else
        return a + w * c;
#endif
    } else return a + w * c;
}
template <class T> FTS_HD cplx<T> cmadd_mi(cplx<T> a, cplx<T> w, cplx<T> c) {       // a + (-i w) c
    if constexpr (sizeof(T) == 8) {
#if defined(__CUDA_ARCH__)
        return mk<T>(fma(w.x, c.y, fma(w.y, c.x, a.x)), fma(-w.x, c.x, fma(w.y, c.y, a.y)));
#else
        const cplx<T> p = w * c; return mk<T>(a.x + p.y, a.y - p.x);
#endif
    } else { const cplx<T> p = w * c; return a + mk<T>(p.y, -p.x); }
}
// (a, c) <- (a + W c, a - W c), W = (MI ? -i : 1) * w
template <bool MI, class T> FTS_HD void bfly_w(cplx<T>& a, cplx<T>& c, cplx<T> w) {
    if constexpr (sizeof(T) == 8) {
        const cplx<T> s = MI ? cmadd_mi(a, w, c) : cmadd(a, w, c);
#if defined(__CUDA_ARCH__)
        c = mk<T>(fma((T)2, a.x, -s.x), fma((T)2, a.y, -s.y));
#else
        c = mk<T>((T)2 * a.x - s.x, (T)2 * a.y - s.y);
#endif
        a = s;
    } else {                                               // complex64: packed pair instructions, 4 per butterfly
        cplx<T> p = w * c;
        if (MI) p = mk<T>(p.y, -p.x);
        c = a - p; a = a + p;
    }
}
// (a, c) <- (a + W c, a - W c), W = exp(-2 pi i M / 16), M = 0..7 at compile time
template <int M, class T> FTS_HD void bfly_c(cplx<T>& a, cplx<T>& c) {
    static_assert(M >= 0 && M < 8, "constant twiddle out of range");
    if constexpr (M == 0) { const cplx<T> s = a + c; c = a - c; a = s; }
    else if constexpr (M == 4) { const cplx<T> p = mk<T>(c.y, -c.x); c = a - p; a = a + p; }
    else if constexpr ((M == 2 || M == 6) && sizeof(T) == 8) {      // h (t1, t2) resp. h (t2, -t1), t1 = c.x + c.y, t2 = c.y - c.x
        constexpr T h = (T)0.70710678118654752440;
        const T t1 = c.x + c.y, t2 = c.y - c.x;
        const T px = M == 2 ? t1 : t2, py = M == 2 ? t2 : -t1;
#if defined(__CUDA_ARCH__)
        c = mk<T>(fma(-h, px, a.x), fma(-h, py, a.y));
        a = mk<T>(fma(h, px, a.x), fma(h, py, a.y));
#else
        c = mk<T>(a.x - h * px, a.y - h * py); a = mk<T>(a.x + h * px, a.y + h * py);
#endif
    } else bfly_w<false>(a, c, mk<T>((T)cos16(M), (T)(-sin16(M))));
}

// multiply by exp(-2 pi i M / 16), M = 0..3 at compile time (general position: 2 mul + 2 fma; M = 2: 2 add + 2 mul)
template <int M, class T> FTS_HD cplx<T> mul_c16(cplx<T> a) {
    if constexpr (M == 0) return a;
    else return mul_w16<M, -1>(a);
}
template <class T> FTS_HD cplx<T> csq(cplx<T> a) { return mk<T>((a.x - a.y) * (a.x + a.y), (T)2 * a.x * a.y); }

// In-register twisted DFT of R points held at v[OFF + S*i].  TWISTED: zp[j] = zeta^(2^j), j = 0..log2(R)-1, for this thread
// and group; level L uses W = zp[log2(R) - L] * exp(-2 pi i (E mod 2^(L-2)) / 2^L) (the constant factor is a 16th root of
// unity applied in registers: shared-memory bandwidth, not the fp64 pipe, bounds the passes, and a 16-byte twiddle load
// costs four wavefronts however many lanes share it).  Otherwise zeta = 1 and every W is known at compile time.
template <int R, int S, int OFF, bool TWISTED, class T, int NV, int NZ>
FTS_HD void tdft_reg(cplx<T> (&v)[NV], const cplx<T> (&zp)[NZ]) {
    if constexpr (R > 1) {
        static_for<1, ilog2(R) + 1>([&](auto ll) {
            constexpr int L = decltype(ll)::value, Rc = R >> (L - 1), half = Rc / 2, Q = L >= 2 ? (1 << (L - 2)) : 1;
            static_for<0, (1 << (L - 1))>([&](auto bb) {
                constexpr int blk = decltype(bb)::value, E = bitrev(blk, L - 1);
                [[maybe_unused]] constexpr bool MI = L >= 2 && E >= Q;
                if constexpr (TWISTED) {
                    const cplx<T> w = mul_c16<((E % Q) * 16) / (1 << L)>(zp[ilog2(R) - L]);
                    static_for<0, half>([&](auto ii) {
                        constexpr int p0 = OFF + S * (blk * Rc + decltype(ii)::value), p1 = p0 + S * half;
                        bfly_w<MI>(v[p0], v[p1], w);
                    });
                } else {
                    static_for<0, half>([&](auto ii) {
                        constexpr int p0 = OFF + S * (blk * Rc + decltype(ii)::value), p1 = p0 + S * half;
                        bfly_c<(E * 16) / (1 << L)>(v[p0], v[p1]);
                    });
                }
            });
        });
        cplx<T> tmp[R];
        static_for<0, R>([&](auto ii) { constexpr int i = decltype(ii)::value; tmp[i] = v[OFF + S * bitrev(i, ilog2(R))]; });
        static_for<0, R>([&](auto ii) { constexpr int i = decltype(ii)::value; v[OFF + S * i] = tmp[i]; });
    }
}

// Factorisation of a pencil of N points over threads holding EPT values each.
template <int N, int EPT>
struct PencilShape {
    static constexpr int TPP = N / EPT;                 // threads per pencil
    static constexpr bool ONE = (TPP == 1);             // whole pencil in one thread
    static constexpr int R1 = ONE ? N : EPT;            // first-stage radix (stride R2 in n)
    static constexpr int R2 = ONE ? 1 : N / R1;         // second-stage radix
    static constexpr int G1 = EPT / R1;                 // first-stage butterflies per thread
    static constexpr int G2 = ONE ? 1 : EPT / R2;       // second-stage butterflies per thread
    static_assert(N % EPT == 0 && R1 * R2 == N && R1 <= 16 && R2 <= 16 && R2 <= EPT, "unsupported pencil shape");
    static_assert(ONE || (TPP * G1 == R2 && TPP * G2 == R1), "inconsistent pencil shape");
};

// Shared-memory addressing of the exchange buffer.  An element of the intermediate Y[n2][k1] of pencil
// `p` (p = pencil slot inside the CTA) lives at  p*PS + k1*ROW + n2*ES  (in complex elements).
//   strided passes (x, y): PS = 1, ES = TZ, ROW = R2*TZ   -> lanes = consecutive pencils, conflict-free
//   contiguous pass (z):   ES = 1, ROW = R2+1, PS = padded pencil stride chosen by the caller
template <int PS_, int ROW_, int ES_> struct XchgLayout { static constexpr int PS = PS_, ROW = ROW_, ES = ES_; };

// Padded pencil stride (in complex elements) of the contiguous-pass exchange buffer: rows of R2+1 (odd), and
// PS = TPP (mod lanes-per-phase) so that the pencils sharing one shared-memory phase hit disjoint banks.
template <class T, int N, int EPT>
constexpr int contig_ps() {
    typedef PencilShape<N, EPT> S;
    constexpr int lpp = 128 / (2 * (int)sizeof(T));       // lanes per shared-memory phase: 8 (complex128) or 16 (complex64)
    int ps = S::R1 * (S::R2 + 1);
    if (S::TPP < lpp) while (ps % lpp != S::TPP % lpp) ++ps;
    return ps;
}

template <class T, int N, int EPT>
struct Pencil {
    typedef PencilShape<N, EPT> S;
    typedef cplx<T> C;

    // forward transform, part A: radix-R1 butterflies + inter-stage twiddle.  The twiddles are stored per
    // (register, thread): tw[r*TPP + t] = exp(-2 pi i (t + TPP*g) k1 / N) with g = r % G1, k1 = r / G1, so that the
    // lanes of a warp read consecutive (contiguous pass) or identical (strided pass) addresses.
    // Inter-stage twiddle of register r (G1 = 1 for every two-stage shape): z^r with z = exp(-2 pi i t / N), stored per
    // (register, thread) at tw[r*TPP + t] so that lanes read consecutive or identical addresses.  Shared memory bandwidth is
    // what bounds the fused passes, so only z, z^2, z^3 and z^4, z^8, z^12 are LOADED (correctly rounded host values); the
    // others are one product z^(4a) * z^b (one extra rounding, < 2 ulp): 9 of 15 loads (3 of 7 for radix 8) become 4 flops each.
    template <int DIR, class TW>
    static FTS_HD void twiddle(C (&v)[EPT], int t, const TW* tw) {
        static_assert(S::ONE || S::G1 == 1, "twiddle scheme assumes one first-stage butterfly per thread");
        if constexpr (!S::ONE) {
            auto get = [&](int r) { TW w = tw[r * S::TPP + t]; return mk<T>((T)w.x, DIR < 0 ? (T)w.y : -(T)w.y); };
            const C w1 = get(1), w2 = get(2), w3 = get(3);
            v[1] = v[1] * w1; v[2] = v[2] * w2; v[3] = v[3] * w3;
            static_for<1, S::R1 / 4>([&](auto aa) {
                constexpr int a = decltype(aa)::value;
                const C wa = get(4 * a);
                v[4 * a] = v[4 * a] * wa;
                v[4 * a + 1] = v[4 * a + 1] * (wa * w1);
                v[4 * a + 2] = v[4 * a + 2] * (wa * w2);
                v[4 * a + 3] = v[4 * a + 3] * (wa * w3);
            });
        }
    }
    // Forward transform with FMA butterflies (see tdft_reg): part A = plain R1-point DFT per thread, no inter-stage
    // multiply; part B (after the same exchange A -> B) = R2-point DFTs twisted by zeta = exp(-2 pi i k1 / N),
    // k1 = t + TPP*g2.  Two twiddles are loaded per group, tw2[k1] = zeta and tw2[R1 + k1] = zeta^TW2_E1 (correctly rounded
    // host values); the other powers zeta^(2^j) are one squaring away.
    static constexpr int LOG2R2 = S::ONE ? 0 : ilog2(S::R2);
    static constexpr int TW2_E1 = S::ONE ? 1 : (S::R2 >= 8 ? S::R2 / 4 : (S::R2 >= 4 ? S::R2 / 2 : 1));
    static FTS_HD void fwd2_a(C (&v)[EPT]) {
        const C one[1] = {mk<T>(1, 0)};
        static_for<0, S::G1>([&](auto g) { tdft_reg<S::R1, S::G1, decltype(g)::value, false>(v, one); });
    }
    template <class TW>
    static FTS_HD void fwd2_b(C (&v)[EPT], int t, const TW* tw2) {
        if constexpr (!S::ONE)
            static_for<0, S::G2>([&](auto g) {
                constexpr int g2 = decltype(g)::value, J1 = ilog2(TW2_E1);
                C zp[LOG2R2 > 0 ? LOG2R2 : 1];
                const TW a = tw2[t + S::TPP * g2];
                zp[0] = mk<T>((T)a.x, (T)a.y);
                if constexpr (J1 > 0 && J1 < LOG2R2) { const TW b = tw2[S::R1 + t + S::TPP * g2]; zp[J1] = mk<T>((T)b.x, (T)b.y); }
                static_for<1, LOG2R2>([&](auto jj) { constexpr int j = decltype(jj)::value; if constexpr (j != J1) zp[j] = csq(zp[j - 1]); });
                tdft_reg<S::R2, S::G2, g2, true>(v, zp);
            });
    }
    // host: angle (in units of 2 pi) of tw2[slot * R1 + k1], slot = 0, 1
    static long double tw2_turns(int slot, int k1) { return -((long double)k1 * (slot ? TW2_E1 : 1) / (long double)N); }
    static constexpr int TW2_SLOTS = S::ONE ? 0 : 2;

    // forward transform, part A: radix-R1 butterflies + inter-stage twiddle.
    template <class TW>
    static FTS_HD void fwd_a(C (&v)[EPT], int t, const TW* tw) {
        static_for<0, S::G1>([&](auto g) { dft_reg<S::R1, S::G1, decltype(g)::value, -1>(v); });
        twiddle<-1>(v, t, tw);
    }
    // exchange A -> B: after store + barrier + load, register g' + G2*n2 of thread t holds Y[n2][k1 = t + TPP*g'].
    template <class L>
    static FTS_HD void xchg_store_a(const C (&v)[EPT], int t, C* sm, int p) {
        if constexpr (!S::ONE)
            static_for<0, EPT>([&](auto rr) {
                constexpr int r = decltype(rr)::value, g = r % S::G1, k1 = r / S::G1;
                sm[p * L::PS + k1 * L::ROW + (t + S::TPP * g) * L::ES] = v[r];
            });
    }
    template <class L>
    static FTS_HD void xchg_load_b(C (&v)[EPT], int t, const C* sm, int p) {
        if constexpr (!S::ONE)
            static_for<0, EPT>([&](auto rr) {
                constexpr int r = decltype(rr)::value, g2 = r % S::G2, n2 = r / S::G2;
                v[r] = sm[p * L::PS + (t + S::TPP * g2) * L::ROW + n2 * L::ES];
            });
    }
    // forward part B: radix-R2 butterflies.  Afterwards register r of thread t holds mode k = t + TPP*r.
    static FTS_HD void fwd_b(C (&v)[EPT]) {
        if constexpr (!S::ONE) static_for<0, S::G2>([&](auto g) { dft_reg<S::R2, S::G2, decltype(g)::value, -1>(v); });
    }
    // inverse = the mirror image: part B (radix-R2), exchange B -> A, part A (conjugate twiddle, radix-R1).
    static FTS_HD void inv_b(C (&v)[EPT]) {
        if constexpr (!S::ONE) static_for<0, S::G2>([&](auto g) { dft_reg<S::R2, S::G2, decltype(g)::value, +1>(v); });
    }
    template <class L>
    static FTS_HD void xchg_store_b(const C (&v)[EPT], int t, C* sm, int p) {
        if constexpr (!S::ONE)
            static_for<0, EPT>([&](auto rr) {
                constexpr int r = decltype(rr)::value, g2 = r % S::G2, n2 = r / S::G2;
                sm[p * L::PS + (t + S::TPP * g2) * L::ROW + n2 * L::ES] = v[r];
            });
    }
    template <class L>
    static FTS_HD void xchg_load_a(C (&v)[EPT], int t, const C* sm, int p) {
        if constexpr (!S::ONE)
            static_for<0, EPT>([&](auto rr) {
                constexpr int r = decltype(rr)::value, g = r % S::G1, k1 = r / S::G1;
                v[r] = sm[p * L::PS + k1 * L::ROW + (t + S::TPP * g) * L::ES];
            });
    }
    template <class TW>
    static FTS_HD void inv_a(C (&v)[EPT], int t, const TW* tw) {
        twiddle<+1>(v, t, tw);
        static_for<0, S::G1>([&](auto g) { dft_reg<S::R1, S::G1, decltype(g)::value, +1>(v); });
    }
};

}  // namespace fts
#endif
