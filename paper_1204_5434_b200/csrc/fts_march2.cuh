// fts_march2.cuh — the contour march for large cubic grids (pencil length 128 or 256):
// ONE persistent kernel per propagator solve, tiles staged by TMA, pencils private to a warp.
//
// The arithmetic is that of fts_march.cuh (same Pencil butterflies) except that the inverse transform is run as
// conj o forward o conj (one transform body, half the code); the two kernels agree to rounding.  What differs is how
// data moves:
//
//   * Every work item moves whole tiles between global memory and shared memory with TMA
//     (cp.async.bulk.tensor on 4-D tensor maps for the strided x / y tiles [N][8 z], 128-byte-swizzled (complex128) or
//     64-byte-swizzled (complex64); plain cp.async.bulk for the contiguous z tiles), issued by one producer thread and
//     one store thread per CTA.  Compute warps never execute a global load, store, atomic, fence or poll.
//   * A pencil of N points is held by TPP = N/16 lanes of ONE warp (16 complex values per lane), so the exchange of
//     the two-stage transform is warp-private: __syncwarp() instead of CTA barriers, and the four compute warps of a
//     CTA drift apart freely (their shared-memory and fp64 phases interleave instead of colliding).
//   * The exchange happens IN PLACE inside the tile buffer the data arrived in (no separate exchange or stash
//     buffers): logical exchange slot (k1, n2) lives in row  k1*R2 + (n2 xor k1)  of the tile, which keeps both
//     access patterns conflict-free under the TMA swizzle and makes every address  base + (V(thread) xor K(register))
//     with compile-time K.  A T item rotates three buffers (H -> q, e4 -> F, F -> H), a Z item two, a Y item one;
//     buffers are allocated round-robin and are released in allocation order.
//   * Dependencies are per yz-plane (Y1 -> Z -> Y2) and per step (T <-> U), so the Y1/Z/Y2 work of a plane runs a
//     few planes behind each other and the plane's F and H stay in L2 between them (HBM sees 11 field transfers per
//     step instead of 17-18).  Tickets are decoded arithmetically; the two propagators' items alternate.
//
// Roles per CTA (192 threads): warps 0-3 compute, warp 4 lane 0 = producer (tickets, dependency polling, TMA loads),
// warp 5 lane 0 = store thread (TMA stores, completion counters, buffer release).
#ifndef FTS_MARCH2_CUH
#define FTS_MARCH2_CUH

#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "fts_march.cuh"

namespace fts {

enum { M2_NBUF = 3, M2_RING = 4, M2_NT = 128, M2_LAUNCH = 192, M2_SEG_SMEM = 224 };
enum { M2_FIRST = 1, M2_FIN = 2, M2_START = 4, M2_RELOAD = 8, M2_JOBH = 16, M2_KEEP = 32, M2_DENS = 64 };
enum { M2_MAP_F = 0, M2_MAP_H = 2, M2_MAP_E = 4, M2_MAP_Q = 8 };     // + propagator (F, H, Q) or factor-field index (E, 0..3)

struct March2Maps {
    CUtensorMap x[10];           // x tiles: box {16 scalars, 1, N, 1} of F0 F1 H0 H1 E0 E1 E2 E3 Q0 Q1
    CUtensorMap y[4];            // y tiles: box {16 scalars, N, 1, 1} of F0 F1 H0 H1
};

struct March2Args {
    void* F[2]; void* H[2]; const void* e4[4];
    const void* tab[3][2];       // per dimension: exp(-k_d^2 ds)/N, exp(-k_d^2 ds/2)/N
    const void* tw;              // twiddles of the twisted second stage, tw2[slot * R1 + k1] (fts_pencil.h)
    int Ns, jA, nspecies, nprop, nsteps, lag, skew;
    const signed char* seg;      // species per contour segment (fts_march.cuh, species_index)
    int packed;                  // N1 real-field fast path: one march of z = q + i q+ (fts_march.cuh, cmul)
    const void* q[2];            // slice stores (the density partner is read straight from global memory)
    DensArgs dens;               // S6: Simpson density sums accumulated by the T items (fts_march.cuh)
    unsigned* ticket;
    unsigned* cnt;               // completion counters [prop][step][2 + 2 N]: T, Y2 (all planes), Y1[plane], Z[plane]
    int* err;
};

struct M2Desc { int kind, flags, b, s, idx, plane, spE, spS; };      // kind < 0: end of march

template <class T, int N>
struct M2Cfg {
    typedef PencilShape<N, 16> S;
    typedef cplx<T> C;
    static constexpr int ES = (int)sizeof(C);
    static constexpr int RB = 8 * ES;                       // bytes of one strided-tile row: 8 z
    static constexpr unsigned SWM = RB == 128 ? 7u : 3u;    // TMA swizzle: 16-byte chunk index ^= (address >> 7) & SWM
    static constexpr int TPP = S::TPP, R2 = S::R2, G2 = S::G2;
    static constexpr int ZPW = 32 / TPP;                    // pencils per warp
    static constexpr int WPT = 8 / ZPW;                     // warps per strided tile
    static constexpr int G = 4 / WPT;                       // strided tiles per item
    static constexpr int PPI = 4 * ZPW;                     // contiguous pencils per item
    static constexpr int TILEB = N * RB;
    // contiguous pencils in shared memory: stride N*ES, plus 64 bytes where a warp's pencils would otherwise fall on the
    // same banks (complex64, N = 128: four 1 KB pencils per warp, 64 bytes per pencil and access)
    static constexpr int PPAD = (ES == 8 && N == 128) ? 64 : 0;
    static constexpr int PSTR = N * ES + PPAD;
    static constexpr int BUFB = 2048 * ES + PPI * PPAD;     // one buffer = one item's tile(s) = 128 threads x 16 values
    static constexpr int NT_X = (N * N / 8) / G;            // items of a T phase
    static constexpr int NY = (N / 8) / G;                  // y items per plane and job
    static constexpr int NZ = N / PPI;                      // z items per plane and job
    static constexpr int NY1 = 2 * NY, NZZ = 2 * NZ, NY2 = NY;
    static constexpr int C2 = 2 + 2 * N;                    // counters per (propagator, step)
    static constexpr size_t SMEM = (size_t)M2_NBUF * BUFB + (size_t)N * ES + (size_t)6 * N * sizeof(T) + 512;
    static_assert(3 * M2_NBUF * 8 + 2 * M2_RING * 8 + M2_RING * 32 + M2_SEG_SMEM <= 512, "control block overflows");
    static_assert(S::G1 == 1 && TPP == R2 && G * TILEB == 2048 * ES && PPI * N * ES == 2048 * ES && BUFB % 1024 == 0, "unsupported shape");
};

__host__ __device__ constexpr unsigned m2_swz(unsigned L, unsigned m) { return L ^ (((L >> 7) & m) << 4); }

// ---- PTX wrappers: mbarrier with transaction bytes, TMA, proxy fences -----------------------------------------
__device__ __forceinline__ unsigned m2_sa(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void m2_expect_tx(uint64_t* b, unsigned bytes) {
    asm volatile("{ .reg .b64 st; mbarrier.arrive.expect_tx.shared.b64 st, [%0], %1; }" ::"r"(m2_sa(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ unsigned long long m2_now_ns() { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
// Waits inside a CTA (TMA completion, hand-offs between the roles) can only fail through a bug; they trap after 10 s
// of wall clock instead of hanging the GPU.
__device__ __forceinline__ void m2_wait(uint64_t* b, unsigned parity, int* err) {
    unsigned ok, tries = 0;
    unsigned long long t0 = 0;
    for (;;) {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                     : "=r"(ok) : "r"(m2_sa(b)), "r"(parity) : "memory");
        if (ok) return;
        if ((++tries & 1023u) == 0) {
            const unsigned long long t = m2_now_ns();
            if (t0 == 0) t0 = t;
            else if (t - t0 > 10000000000ull) { atomicExch(err, 2); __trap(); }
        }
    }
}
__device__ __forceinline__ void m2_fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void m2_fence_async() { asm volatile("fence.proxy.async;" ::: "memory"); }
__device__ __forceinline__ void m2_tma_load4(void* dst, const CUtensorMap* map, int c0, int c1, int c2, int c3, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                 ::"r"(m2_sa(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(m2_sa(bar)) : "memory");
}
__device__ __forceinline__ void m2_tma_store4(const CUtensorMap* map, int c0, int c1, int c2, int c3, const void* src) {
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.tile.bulk_group [%0, {%1, %2, %3, %4}], [%5];"
                 ::"l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(m2_sa(src)) : "memory");
}
__device__ __forceinline__ void m2_bulk_load(void* dst, const void* src, unsigned bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(m2_sa(dst)), "l"(src), "r"(bytes), "r"(m2_sa(bar)) : "memory");
}
__device__ __forceinline__ void m2_bulk_store(void* dst, const void* src, unsigned bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(m2_sa(src)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void m2_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void m2_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void m2_wait_all0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

// ---- ticket -> item (arithmetic; the same function serves the host for the totals) ----------------------------
// Round j:  T(q, j) | slots i = 0 .. N+2L+D-1: [Y1(q+,i) Y1(q,i-D) Z(q+,i-L) Z(q,i-D-L) Y2(q+,i-2L) Y2(q,i-D-2L)] | T(q+, j)
// where the q+ items of the slots belong to step j-1 (they run half a step behind) and q's planes trail q+'s by the
// skew D, so that every whole-field dependency (T -> Y1 of the same step, Y2 -> T of the next) is separated by work of
// the other propagator: the first D slots hold only q+ items, the last D only q items.
template <class T, int N>
struct M2Sched {
    typedef M2Cfg<T, N> Cfg;
    int nprop, lag, skew, nsteps, slot_sz, nslots, per_round;
    __host__ __device__ M2Sched(int nprop_, int lag_, int skew_, int nsteps_) : nprop(nprop_), lag(lag_), skew(nprop_ == 2 ? skew_ : 0), nsteps(nsteps_) {
        slot_sz = nprop * (Cfg::NY1 + Cfg::NZZ + Cfg::NY2);
        nslots = N + 2 * lag + skew;
        per_round = nprop * Cfg::NT_X + nslots * slot_sz;
    }
    __host__ __device__ long long total() const { return (long long)(nsteps + 1) * per_round; }
    // returns false for a ticket that carries no work
    __device__ bool decode(unsigned tk, M2Desc& d) const {
        const int round = (int)(tk / (unsigned)per_round);
        int off = (int)(tk % (unsigned)per_round);
        d.flags = 0; d.plane = 0;
        if (off < Cfg::NT_X) { d.kind = PH_T; d.b = 0; d.s = round; d.idx = off; return true; }
        off -= Cfg::NT_X;
        if (off < nslots * slot_sz) {
            const int slot = off / slot_sz; int w = off % slot_sz;
            const int sz[3] = {Cfg::NY1, Cfg::NZZ, Cfg::NY2};
            int kind = 0;
            for (; kind < 3; ++kind) { if (w < nprop * sz[kind]) break; w -= nprop * sz[kind]; }
            const int first = nprop == 2 ? 1 : 0;                   // the propagator listed first in each group
            const int b = w < sz[kind] ? first : 0;
            if (w >= sz[kind]) w -= sz[kind];
            d.kind = PH_Y1 + kind; d.b = b; d.s = round - (nprop == 2 && b == 1 ? 1 : 0);
            d.plane = slot - kind * lag - (nprop == 2 && b == 0 ? skew : 0);
            if (kind < 2) { const int half = sz[kind] / 2; if (w >= half) { d.flags |= M2_JOBH; w -= half; } } else d.flags |= M2_JOBH;
            d.idx = w;
            return d.plane >= 0 && d.plane < N && d.s >= 0 && d.s < nsteps;
        }
        off -= nslots * slot_sz;
        d.kind = PH_T; d.b = 1; d.s = round; d.idx = off;
        return true;
    }
};


__device__ __forceinline__ double flip_sign(double x) { return __hiloint2double(__double2hiint(x) ^ (int)0x80000000, __double2loint(x)); }
__device__ __forceinline__ float flip_sign(float x) { return __int_as_float(__float_as_int(x) ^ (int)0x80000000); }

// Per-thread view of a tile buffer: natural-layout access and the in-place diffusion (see the header).
//   strided tile  (x, y passes): element (row rho, z) at  rho*RB + z*ES, 16-byte chunk index ^= (rho*RB >> 7) & SWM  (TMA swizzle)
//   contiguous tile (z pass):    element i of pencil p at (p*N + i)*ES, no swizzle
// natural layout:   register r <-> point  t + TPP r                      -> address  VA + r*TPP*stride           (additive)
// exchange slot (k1, n2) lives at index  k1*R2 + (n2 ^ (k1 mod R2)):
//   pattern A (k1 = r, n2 = t):            VA ^ K_A(r),  K_A(r) = (r*R2 + (r mod R2)) * stride
//   pattern B (k1 = t + R2 g2, n2 = r/G2): VB ^ K_B(r),  K_B(r) = ((r mod G2)*R2*R2 + r/G2) * stride,  VB from index t*R2 + t
template <class T, int N>
struct M2Lane {
    typedef M2Cfg<T, N> Cfg;
    typedef Pencil<T, N, 16> P;
    typedef cplx<T> C;
    unsigned VAs, VBs, VAc, VBc;         // thread part of the address inside a tile / a pencil
    unsigned offs, offc;                 // this warp's strided sub-tile / this lane's contiguous pencil inside a buffer
    int t;
    const C* s_tw;
    static constexpr int TPP = Cfg::TPP, R2 = Cfg::R2, G2 = Cfg::G2, ES = Cfg::ES, RB = Cfg::RB;
    template <bool CONTIG> static constexpr unsigned stride() { return CONTIG ? (unsigned)ES : (unsigned)RB; }
    template <bool CONTIG> static constexpr unsigned KA(int r) { return m2_swz((unsigned)(r * R2 + (r & (R2 - 1))) * stride<CONTIG>(), CONTIG ? 0u : Cfg::SWM); }
    template <bool CONTIG> static constexpr unsigned KB(int r) { return m2_swz((unsigned)((r % G2) * R2 * R2 + r / G2) * stride<CONTIG>(), CONTIG ? 0u : Cfg::SWM); }
    static __device__ __forceinline__ C ld(const unsigned char* p) { return *reinterpret_cast<const C*>(p); }
    static __device__ __forceinline__ void st(unsigned char* p, C v) { *reinterpret_cast<C*>(p) = v; }

    // Loads are issued in the order the first butterfly level consumes them (pairs r, r + 8), so that the butterflies start
    // after two loads instead of nine.
    template <int G> static constexpr int ld_order(int i) { return G == 1 ? ((i & 1) ? i / 2 + 8 : i / 2) : (i / 8 + 2 * ((i % 8) / 2) + 8 * (i & 1)); }
    template <bool CONTIG> __device__ __forceinline__ void load_nat(C (&v)[16], const unsigned char* base) const {
        const unsigned char* p = base + (CONTIG ? offc + VAc : offs + VAs);
        static_for<0, 16>([&](auto rr) { constexpr int r = ld_order<1>(decltype(rr)::value); v[r] = ld(p + r * TPP * stride<CONTIG>()); });
    }
    template <bool CONTIG> __device__ __forceinline__ void store_nat(const C (&v)[16], unsigned char* base) const {
        unsigned char* p = base + (CONTIG ? offc + VAc : offs + VAs);
        static_for<0, 16>([&](auto rr) { constexpr int r = decltype(rr)::value; st(p + r * TPP * stride<CONTIG>(), v[r]); });
    }
    // exp(a ds d^2/dx_d^2) along the pencil: forward transform, real table (1/N folded in), inverse transform; the two
    // exchanges of each direction happen in place inside `base`.  Every lane of the warp must have consumed whatever the
    // buffer held before the call (first __syncwarp); on return all lanes have finished reading it (last __syncwarp).
    template <bool CONTIG> __device__ __forceinline__ void xst_a(const C (&v)[16], unsigned char* base) const {
        const unsigned va = CONTIG ? VAc : VAs; base += CONTIG ? offc : offs;
        static_for<0, 16>([&](auto rr) { constexpr int r = decltype(rr)::value; st(base + (va ^ KA<CONTIG>(r)), v[r]); });
    }
    template <bool CONTIG> __device__ __forceinline__ void xld_a(C (&v)[16], const unsigned char* base) const {
        const unsigned va = CONTIG ? VAc : VAs; base += CONTIG ? offc : offs;
        static_for<0, 16>([&](auto rr) { constexpr int r = decltype(rr)::value; v[r] = ld(base + (va ^ KA<CONTIG>(r))); });
    }
    template <bool CONTIG> __device__ __forceinline__ void xst_b(const C (&v)[16], unsigned char* base) const {
        const unsigned vb = CONTIG ? VBc : VBs; base += CONTIG ? offc : offs;
        static_for<0, 16>([&](auto rr) { constexpr int r = decltype(rr)::value; st(base + (vb ^ KB<CONTIG>(r)), v[r]); });
    }
    template <bool CONTIG> __device__ __forceinline__ void xld_b(C (&v)[16], const unsigned char* base) const {
        const unsigned vb = CONTIG ? VBc : VBs; base += CONTIG ? offc : offs;
        static_for<0, 16>([&](auto rr) { constexpr int r = ld_order<G2>(decltype(rr)::value); v[r] = ld(base + (vb ^ KB<CONTIG>(r))); });
    }
    // exp(a ds d^2/dx_d^2) along the pencil = F^-1 [table] F, with the inverse transform run as conj o F o conj, so that ONE
    // forward-transform body (radix-R1 butterflies, twiddles, exchange A -> B, radix-R2 butterflies) is executed twice in a
    // rolled loop: the hot code of the kernel is then about 9 KB.  The four compute warps of a CTA run at different places
    // of the kernel, so its working set has to fit the instruction caches (measured: 17 % of the warps' time went to
    // instruction fetch with both transforms unrolled).  The butterflies are shared by the two layouts; only the exchange
    // accesses are specialised.  The real table carries 1/N; conj(v * tab) = (v.x tab, v.y (-tab)).
    __device__ __forceinline__ void diffuse(C (&v)[16], unsigned char* base, bool contig, const T* tab) const {
#pragma unroll 1
        for (int pass = 0; pass < 2; ++pass) {
            P::fwd2_a(v);
            __syncwarp();                                  // every lane has consumed what the buffer held / its B-pattern loads
            if (contig) xst_a<true>(v, base); else xst_a<false>(v, base);
            __syncwarp();
            if (contig) xld_b<true>(v, base); else xld_b<false>(v, base);
            P::fwd2_b(v, t, s_tw);
            if (pass == 0) {
#pragma unroll
                for (int r = 0; r < 16; ++r) { const T w = tab[t + TPP * r]; v[r] = mk<T>(v[r].x * w, v[r].y * (-w)); }
            } else {
#pragma unroll
                for (int r = 0; r < 16; ++r) v[r].y = flip_sign(v[r].y);      // integer pipe: the fp64 pipe is the bound
            }
        }
        __syncwarp();                                      // all exchange reads done before anyone writes natural positions
    }
};

template <class T, int N>
__global__ void __launch_bounds__(M2_LAUNCH, (sizeof(T) == 8 ? 2 : 4)) march2_kernel(const __grid_constant__ March2Maps maps, const March2Args A) {
    typedef M2Cfg<T, N> Cfg;
    typedef Pencil<T, N, 16> P;
    typedef cplx<T> C;
    constexpr int TPP = Cfg::TPP, R2 = Cfg::R2, ES = Cfg::ES, RB = Cfg::RB, BUFB = Cfg::BUFB;
    constexpr unsigned SWM = Cfg::SWM;
    constexpr unsigned TILE2 = 2048 * ES;                                // bytes one item moves per buffer

    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char* s_buf = smem;
    C* s_tw = reinterpret_cast<C*>(smem + M2_NBUF * BUFB);
    T* s_tab = reinterpret_cast<T*>(s_tw + N);                       // [dim][full, half][N]
    unsigned char* ctrl = reinterpret_cast<unsigned char*>(s_tab + 6 * N);
    uint64_t* b_full = reinterpret_cast<uint64_t*>(ctrl);            // [3] tile landed (TMA complete_tx, or a plain arrive)
    uint64_t* b_out = b_full + M2_NBUF;                              // [3] compute threads are done with the buffer (128 arrivals)
    uint64_t* b_free = b_out + M2_NBUF;                              // [3] store thread has released the buffer
    uint64_t* b_ifull = b_free + M2_NBUF;                            // [4] item descriptor published
    uint64_t* b_iempty = b_ifull + M2_RING;                          // [4] descriptor no longer needed (4 warps + store thread)
    M2Desc* s_desc = reinterpret_cast<M2Desc*>(b_iempty + M2_RING);  // [4]
    signed char* s_seg = reinterpret_cast<signed char*>(s_desc + M2_RING);      // species per contour segment, for the producer's lookups; inside the 512-byte control block
                                                                     // (complex128 at N = 256 fits two CTAs per SM with 0.5 KB to spare: no static shared memory)

    const int tid = threadIdx.x;
    for (int i = tid; i < N; i += M2_LAUNCH) s_tw[i] = static_cast<const C*>(A.tw)[i];      // tw2 layout (Pencil::fwd2_b), N/2 entries used
    for (int i = tid; i < 6 * N; i += M2_LAUNCH) s_tab[i] = static_cast<const T*>(A.tab[i / (2 * N)][(i / N) & 1])[i % N];
    const bool seg_in_smem = A.Ns <= M2_SEG_SMEM;
    if (seg_in_smem && A.nspecies == 2) for (int i = tid; i < A.Ns; i += M2_LAUNCH) s_seg[i] = A.seg[i];
    const signed char* const seg = seg_in_smem ? s_seg : A.seg;
    if (tid == 0) {
        for (int i = 0; i < M2_NBUF; ++i) { mbar_init(&b_full[i], 1); mbar_init(&b_out[i], M2_NT); mbar_init(&b_free[i], 1); }
        for (int i = 0; i < M2_RING; ++i) { mbar_init(&b_ifull[i], 1); mbar_init(&b_iempty[i], 5); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const M2Sched<T, N> sched(A.nprop, A.lag, A.skew, A.nsteps);
    auto species = [&](int b, int step) -> int { return species_index(A.packed, A.nspecies, seg, A.Ns, b, step); };      // O5 / O6 block schedule
    const bool cw = A.packed != 0;
    auto nbuf_of = [](int kind) { return kind == PH_T ? 3 : (kind == PH_Z ? 2 : 1); };
    // TMA coordinates of sub-tile g of a strided item (c0 in scalars), and the byte offset of a z item inside a field
    auto xcoord = [](int idx, int g, int& c0, int& c1) { const int tile = idx * Cfg::G + g; c0 = (tile % (N / 8)) * 16; c1 = tile / (N / 8); };
    auto zoffset = [](int plane, int idx) { return ((size_t)plane * N + (size_t)idx * Cfg::PPI) * N * ES; };

    if (tid >= M2_NT) {
        const int role = (tid - M2_NT) >> 5;
        if ((tid & 31) != 0) return;
        if (role == 0) {
            // ===================== producer: tickets, dependencies, TMA loads =====================
            const unsigned total = (unsigned)sched.total();
            unsigned alloc = 0, item = 0;
            const unsigned* dep_ok = nullptr;
            unsigned tk = atomicAdd(A.ticket, 1u);
            bool aborted = false;
            for (;;) {
                M2Desc d;
                bool live = false;
                while (tk < total && !(live = sched.decode(tk, d))) tk = atomicAdd(A.ticket, 1u);
                if (!live) break;
                const unsigned tk_next = atomicAdd(A.ticket, 1u);          // drawn one ahead
                // dependency: the phase this item consumes; it precedes the item in ticket order
                unsigned* cb = A.cnt + ((size_t)d.b * (A.Ns + 1) + d.s) * Cfg::C2;
                const unsigned* dep = nullptr; unsigned need = 0;
                if (d.kind == PH_T) { if (d.s > 0) { dep = cb - Cfg::C2 + 1; need = (unsigned)N * Cfg::NY2; } }
                else if (d.kind == PH_Y1) { dep = cb; need = Cfg::NT_X; }
                else if (d.kind == PH_Z) { dep = cb + 2 + d.plane; need = Cfg::NY1; }
                else { dep = cb + 2 + N + d.plane; need = Cfg::NZZ; }
#ifdef FTS_M2_NODEPS
                dep = nullptr;                                             // measurement build only: wrong results, shows what the schedule costs
#endif
                // T items that accumulate densities read a slice stored by the other propagator's T phase of step Ns - s (one
                // propagator: its own); that phase lies at least a step back in ticket order
                const unsigned* dep2 = nullptr;
                if (d.kind == PH_T && A.dens.on) {
                    const bool two = A.nprop == 2;
                    if (two ? (d.b == 0 ? d.s > A.dens.half : d.s >= A.dens.half) : d.s >= A.dens.half) {
                        d.flags |= M2_DENS;
                        if (!(!two && d.s == A.dens.half)) dep2 = A.cnt + ((size_t)(two ? 1 - d.b : 0) * (A.Ns + 1) + (A.Ns - d.s)) * Cfg::C2;
                    }
                }
                if (d.kind == PH_T && (d.s <= A.dens.keep || d.s == A.nsteps)) d.flags |= M2_KEEP;
#ifdef FTS_M2_NODEPS
                dep2 = nullptr;
#endif
                if (dep2) {
                    unsigned spins = 0;
                    unsigned long long t0 = 0;
                    while (ld_relaxed(dep2) < (unsigned)Cfg::NT_X) {
                        if ((++spins & 4095u) == 0) {
                            const unsigned long long t = m2_now_ns();
                            if (t0 == 0) t0 = t; else if (t - t0 > 5000000000ull) { aborted = true; break; }
                        }
                        __nanosleep(20);
                    }
                    if (aborted) { atomicExch(A.err, 1); break; }
                    if (!dep || dep == dep_ok) fence_acquire();
                }
                if (dep && dep != dep_ok) {
                    unsigned spins = 0;
                    unsigned long long t0 = 0;
                    while (ld_relaxed(dep) < need) {                       // another CTA's work: give up after 5 s and drain (never hang the GPU)
                        if ((++spins & 4095u) == 0) {
                            const unsigned long long t = m2_now_ns();
                            if (t0 == 0) t0 = t; else if (t - t0 > 5000000000ull) { aborted = true; break; }
                        }
                        __nanosleep(20);
                    }
                    if (aborted) { atomicExch(A.err, 1); break; }
                    fence_acquire();
                    dep_ok = dep;
                }
                m2_fence_async();                                          // generic-proxy acquire -> async-proxy loads
                if (d.kind == PH_T) {
                    d.flags |= (d.s == 0 ? M2_FIRST : M2_FIN) | (d.s < A.nsteps ? M2_START : 0);
                    d.spE = species(d.b, d.s > 0 ? d.s - 1 : 0); d.spS = species(d.b, d.s);
                    if (d.s > 0 && d.s < A.nsteps && d.spE != d.spS) d.flags |= M2_RELOAD;
                    if (d.s == 0) d.spE = d.spS;
                } else d.spE = d.spS = species(d.b, d.s);
                const int slot = item % M2_RING;
                if (item >= M2_RING) m2_wait(&b_iempty[slot], ((item / M2_RING) - 1) & 1, A.err);
                s_desc[slot] = d;
                const int nb = nbuf_of(d.kind);
                for (int k = 0; k < nb; ++k, ++alloc) {
                    const int buf = alloc % M2_NBUF; const unsigned use = alloc / M2_NBUF;
                    if (use > 0) m2_wait(&b_free[buf], (use - 1) & 1, A.err);
                    unsigned char* dst = s_buf + buf * BUFB;
                    if (d.kind == PH_T) {
                        // buffers: 0 = H (-> q), 1 = e4 (-> F), 2 = F (-> H).  First step: only e4 is loaded.
                        const bool load = k == 1 ? true : !(d.flags & M2_FIRST);
                        if (!load) mbar_arrive(&b_full[buf]);
                        else {
                            m2_expect_tx(&b_full[buf], TILE2);
                            const CUtensorMap* mp = &maps.x[k == 0 ? M2_MAP_H + d.b : (k == 1 ? M2_MAP_E + d.spE : M2_MAP_F + d.b)];
                            for (int g = 0; g < Cfg::G; ++g) { int c0, c1; xcoord(d.idx, g, c0, c1); m2_tma_load4(dst + g * Cfg::TILEB, mp, c0, c1, 0, 0, &b_full[buf]); }
                        }
                    } else if (d.kind == PH_Z) {
                        m2_expect_tx(&b_full[buf], TILE2);
                        const char* src = k == 0 ? static_cast<const char*>((d.flags & M2_JOBH) ? A.H[d.b] : A.F[d.b]) : static_cast<const char*>(A.e4[d.spE]);
                        if constexpr (Cfg::PPAD == 0) m2_bulk_load(dst, src + zoffset(d.plane, d.idx), TILE2, &b_full[buf]);
                        else for (int p = 0; p < Cfg::PPI; ++p) m2_bulk_load(dst + p * Cfg::PSTR, src + zoffset(d.plane, d.idx) + (size_t)p * N * ES, N * ES, &b_full[buf]);
                    } else {
                        m2_expect_tx(&b_full[buf], TILE2);
                        const CUtensorMap* mp = &maps.y[((d.flags & M2_JOBH) ? 2 : 0) + d.b];
                        for (int g = 0; g < Cfg::G; ++g) m2_tma_load4(dst + g * Cfg::TILEB, mp, (d.idx * Cfg::G + g) * 16, 0, d.plane, 0, &b_full[buf]);
                    }
                    if (k == 0) mbar_arrive(&b_ifull[slot]);               // publish as soon as the primary tile is on its way
                }
                ++item;
                tk = tk_next;
            }
            // end of march (or abort): sentinel for the compute warps and the store thread
            const int slot = item % M2_RING;
            if (item >= M2_RING) m2_wait(&b_iempty[slot], ((item / M2_RING) - 1) & 1, A.err);
            s_desc[slot].kind = -1;
            mbar_arrive(&b_ifull[slot]);
            return;
        }
        // ===================== store thread: TMA stores, completion counters, buffer release =====================
        unsigned alloc = 0;
        for (unsigned item = 0;; ++item) {
            const int slot = item % M2_RING;
            m2_wait(&b_ifull[slot], (item / M2_RING) & 1, A.err);
            const volatile M2Desc* dv = &s_desc[slot];
            M2Desc d;
            d.kind = dv->kind; d.flags = dv->flags; d.b = dv->b; d.s = dv->s; d.idx = dv->idx; d.plane = dv->plane; d.spE = dv->spE; d.spS = dv->spS;
            if (d.kind < 0) break;
            const int nb = nbuf_of(d.kind);
            unsigned* cb = A.cnt + ((size_t)d.b * (A.Ns + 1) + d.s) * Cfg::C2;
            for (int k = 0; k < nb; ++k, ++alloc) {
                const int buf = alloc % M2_NBUF; const unsigned use = alloc / M2_NBUF;
                m2_wait(&b_out[buf], use & 1, A.err);
                const unsigned char* src = s_buf + buf * BUFB;
                bool store = true;
                if (d.kind == PH_T) {
                    if (k > 0 && !(d.flags & M2_START)) store = false;
                    if (k == 0 && !(d.flags & M2_KEEP)) store = false;            // meet-in-the-middle: this slice is not retained
                    if (store) {
                        const CUtensorMap* mp = &maps.x[k == 0 ? M2_MAP_Q + d.b : (k == 1 ? M2_MAP_F + d.b : M2_MAP_H + d.b)];
                        const int c3 = k == 0 ? slice_slot(d.s, A.dens.keep) : 0;
                        for (int g = 0; g < Cfg::G; ++g) { int c0, c1; xcoord(d.idx, g, c0, c1); m2_tma_store4(mp, c0, c1, 0, c3, src + g * Cfg::TILEB); }
                    }
                } else if (d.kind == PH_Z) {
                    if (k == 1) store = false;
                    else {
                        char* dst = static_cast<char*>((d.flags & M2_JOBH) ? A.H[d.b] : A.F[d.b]) + zoffset(d.plane, d.idx);
                        if constexpr (Cfg::PPAD == 0) m2_bulk_store(dst, src, TILE2);
                        else for (int p = 0; p < Cfg::PPI; ++p) m2_bulk_store(dst + (size_t)p * N * ES, src + p * Cfg::PSTR, N * ES);
                    }
                } else {
                    const CUtensorMap* mp = &maps.y[((d.flags & M2_JOBH) ? 2 : 0) + d.b];
                    for (int g = 0; g < Cfg::G; ++g) m2_tma_store4(mp, (d.idx * Cfg::G + g) * 16, 0, d.plane, 0, src + g * Cfg::TILEB);
                }
                if (store) { m2_commit(); m2_wait_read0(); }
                mbar_arrive(&b_free[buf]);
                if (k == nb - 1) {                                         // the item's last buffer: all its stores are complete -> signal
                    m2_wait_all0();
                    m2_fence_async();
                    __threadfence();
                    unsigned* c = d.kind == PH_T ? cb : d.kind == PH_Y2 ? cb + 1 : d.kind == PH_Y1 ? cb + 2 + d.plane : cb + 2 + N + d.plane;
                    atomicAdd(c, 1u);
                }
            }
            mbar_arrive(&b_iempty[slot]);
        }
        return;
    }

    // ===================== compute warps =====================
    const int lane = tid & 31, w = tid >> 5;
    const int t = lane % TPP, zz = lane / TPP;
    // strided tiles: sub-tile g = w / WPT, z = (w % WPT) * ZPW + zz; contiguous: pencil p = w * ZPW + zz
    const unsigned vs_l = (unsigned)(t * RB + ((w % Cfg::WPT) * Cfg::ZPW + zz) * ES);
    const unsigned sub = (unsigned)((w / Cfg::WPT) * Cfg::TILEB);
    const unsigned VAs = m2_swz(vs_l, SWM), VBs = m2_swz((unsigned)((t * R2 + t) * RB) + (vs_l & (RB - 1)), SWM);
    const unsigned pen = (unsigned)((w * Cfg::ZPW + zz) * Cfg::PSTR);
    const unsigned VAc = t * ES, VBc = (t * R2 + t) * ES;

    const M2Lane<T, N> L = {VAs, VBs, VAc, VBc, sub, pen, t, s_tw};
    auto load_nat = [&](C (&v)[16], const unsigned char* base, bool contig) { if (contig) L.template load_nat<true>(v, base); else L.template load_nat<false>(v, base); };
    auto store_nat = [&](const C (&v)[16], unsigned char* base, bool contig) { if (contig) L.template store_nat<true>(v, base); else L.template store_nat<false>(v, base); };
    auto diffuse = [&](C (&v)[16], unsigned char* base, bool contig, const T* tab) { L.diffuse(v, base, contig, tab); };
    // this thread is done with the buffer; `stored`: it wrote a tile the store thread will hand to TMA (generic -> async proxy)
    auto release = [&](int buf, bool stored) { if (stored) m2_fence_async_smem(); mbar_arrive(&b_out[buf]); };

    // One item = a short program of stages  [load tile ->] diffuse -> post action.  The loop below has ONE call site of
    // load_nat / diffuse / store_nat (two bodies each: strided and contiguous layout), which keeps the kernel's hot code
    // small enough for the instruction caches although the four warps of a CTA run at different places of it.
    unsigned alloc = 0;
    for (unsigned item = 0;; ++item) {
        const int slot = item % M2_RING;
        m2_wait(&b_ifull[slot], (item / M2_RING) & 1, A.err);
        const volatile M2Desc* dv = &s_desc[slot];
        const int kind = dv->kind, flags = dv->flags;
        if (kind < 0) break;
        const int bA = alloc % M2_NBUF, bB = (alloc + 1) % M2_NBUF, bC = (alloc + 2) % M2_NBUF;
        const unsigned uA = alloc / M2_NBUF, uB = (alloc + 1) / M2_NBUF, uC = (alloc + 2) / M2_NBUF;
        unsigned char* pA = s_buf + bA * BUFB; unsigned char* pB = s_buf + bB * BUFB; unsigned char* pC = s_buf + bC * BUFB;
        const bool contig = kind == PH_Z, jobh = flags & M2_JOBH;
        const T* tabd = s_tab + (kind == PH_T ? 0 : (contig ? 4 * N : 2 * N));      // [full][half] of the item's dimension
        alloc += kind == PH_T ? 3 : (contig ? 2 : 1);
        C v[16];
        // q_s = (4 e4 Dx'[H] - F)/3 -> slice (Eq. 12);  start of step s: stash e4 q_s, v = e4^2 q_s.
        // Buffers of a T item: A = H (then q_s), B = e4 (then F), C = F (then the stash, then H).
        // element r of this thread inside a field (x tiles): gbase_of() + r TPP N^2
        auto gbase_of = [&]() {
            const int tile = dv->idx * Cfg::G + w / Cfg::WPT, z = (tile % (N / 8)) * 8 + (w % Cfg::WPT) * Cfg::ZPW + zz, iy = tile / (N / 8);
            return (t * N + iy) * N + z;
        };
        // S6 (Eq. 8, DensArgs): the slice just formed (re-read from the tile at pq) times the stored partner slice,
        // Simpson-weighted, into the sums.  Partner and sums are read straight from global memory (prefetched into L2 when the
        // item started), four elements per round trip: all loads of a batch are issued before its first store.
        auto accumulate_density = [&](const unsigned char* pq) {
            const int b = dv->b, s = dv->s; const bool two = A.nprop == 2;
            const int jp = (two && b == 1) ? A.Ns - s : s;
            const bool self = !two && s == A.dens.half;
            T wA = (T)A.dens.cA[jp], wB = (T)A.dens.cB[jp], wA2 = 0, wB2 = 0;
            if (cw) { if (!self) { wA2 = (T)A.dens.cA[A.Ns - jp]; wB2 = (T)A.dens.cB[A.Ns - jp]; } }
            else if (!two && !self) wA += (T)A.dens.cA[A.Ns - jp];
            const int gb = gbase_of();
            const C* partner = static_cast<const C*>(A.q[two ? 1 - b : 0]) + (size_t)(A.Ns - s) * N * N * N + gb;
            for (int pass = 0; pass < 2; ++pass) {                      // sums of species A, then B (both only at the block junction)
                const T w1 = pass == 0 ? wA : wB;
                if (cw ? pass == 1 : w1 == (T)0) continue;
                C* acc = static_cast<C*>(A.dens.acc[b][cw ? 0 : pass]) + gb;
#pragma unroll 1
                for (int r0 = 0; r0 < 16; r0 += 4) {
                    C zp[4], a[4], q[4];
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        const int off = (r0 + k) * TPP * N * N;
                        q[k] = L.ld(pq + (r0 + k) * TPP * RB);
                        zp[k] = self ? q[k] : ldcg(partner + off);
                        a[k] = ldcg(acc + off);
                    }
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        const int off = (r0 + k) * TPP * N * N;
                        if (cw) {                                       // z = q + i q+: pairs (s, Ns-s) and (Ns-s, s); sums (A, B) as (re, im)
                            const T p1 = q[k].x * zp[k].y, p2 = zp[k].x * q[k].y;
                            stcg(acc + off, mk<T>(a[k].x + wA * p1 + wA2 * p2, a[k].y + wB * p1 + wB2 * p2));
                        } else {
                            const C pr = q[k] * zp[k];
                            stcg(acc + off, mk<T>(a[k].x + w1 * pr.x, a[k].y + w1 * pr.y));
                        }
                    }
                }
            }
        };
        // L2 prefetch of what accumulate_density will read (issued when the item starts, a transform ahead of its use)
        auto prefetch_density = [&]() {
            if ((zz & 1) != 0) return;
            const int b = dv->b, s = dv->s; const bool two = A.nprop == 2;
            const int gb = gbase_of();
            const C* partner = static_cast<const C*>(A.q[two ? 1 - b : 0]) + (size_t)(A.Ns - s) * N * N * N + gb;
            const int jp = (two && b == 1) ? A.Ns - s : s;
            const C* acc = static_cast<const C*>(A.dens.acc[b][(cw || A.dens.cA[jp] != 0.0) ? 0 : 1]) + gb;
#pragma unroll 4
            for (int r = 0; r < 16; ++r) {
                asm volatile("prefetch.global.L2 [%0];" ::"l"(partner + r * TPP * N * N));
                asm volatile("prefetch.global.L2 [%0];" ::"l"(acc + r * TPP * N * N));
            }
        };
        auto combine = [&]() {
            m2_wait(&b_full[bB], uB & 1, A.err);
            m2_wait(&b_full[bC], uC & 1, A.err);
            const bool fin = flags & M2_FIN, start = flags & M2_START, reload = flags & M2_RELOAD;
            const unsigned char* pe = pB + sub + VAs; const unsigned char* pf = pC + sub + VAs;
            unsigned char* pq = pA + sub + VAs; unsigned char* ph = pC + sub + VAs;
            const bool dens = flags & M2_DENS;
            const C* e4s = nullptr; int gbase = 0;
            if (reload) { gbase = gbase_of(); e4s = static_cast<const C*>(A.e4[dv->spS]); }      // block junction: the new species' factors straight from global memory
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                C e = L.ld(pe + r * TPP * RB);
                if (fin) {
                    const C f = L.ld(pf + r * TPP * RB);
                    const C h = cmul(v[r], e, cw);
                    v[r] = mk<T>(((T)4 * h.x - f.x) * (T)(1.0 / 3.0), ((T)4 * h.y - f.y) * (T)(1.0 / 3.0));
                } else v[r] = mk<T>(1, cw ? 1 : 0);                              // q(x,0) = 1, q+(x,s=1) = 1
                L.st(pq + r * TPP * RB, v[r]);
                if (start) {
                    if (reload) e = ldcg(e4s + gbase + r * TPP * N * N);
                    const C hb = cmul(v[r], e, cw);
                    L.st(ph + r * TPP * RB, hb);
                    v[r] = cmul(hb, e, cw);
                }
            }
            if (dens) accumulate_density(pq);
            release(bA, true);                                          // q_s -> slice store
            if (!start) { release(bB, false); release(bC, false); }
            return start;
        };
        if (kind == PH_T && (flags & M2_DENS)) prefetch_density();
        m2_wait(&b_full[bA], uA & 1, A.err);
        unsigned char* cur = pA; int curb = bA;
        const T* tab = (kind == PH_T || jobh) ? tabd + N : tabd;
        int st = 0;
        bool run = true, need_load = true;
        if (kind == PH_T && !(flags & M2_FIN)) {                            // first slice: nothing to finish
            run = combine();
            cur = pB; curb = bB; tab = tabd; st = 1; need_load = false;
        }
#pragma unroll 1
        while (run) {
            if (need_load) load_nat(v, cur, contig);
#ifdef FTS_M2_SYNC_WARPS
            bar_compute<M2_NT>();
#endif
            diffuse(v, cur, contig, tab);
            bool store = true;
            if (kind == PH_T) {
                if (st == 0) {                                              // H' = Dx'[H] done
                    store = false;
                    run = combine();
                    cur = pB; curb = bB; tab = tabd; st = 1; need_load = false;      // next: F = Dx[e2 q_s], exchanged inside the e4 buffer
                } else if (st == 2) run = false;                            // H = Dx'[e4 q_s] done
            } else if (contig) {
                if (st == 0) {                                              // F = e2 Dz F;  H = Dz'[e2 Dz' H]
                    m2_wait(&b_full[bB], uB & 1, A.err);
#pragma unroll
                    for (int r = 0; r < 16; ++r) { const C e = L.ld(pB + pen + VAc + r * TPP * ES); v[r] = cmul(v[r], cmul(e, e, cw), cw); }
                    if (jobh) { store = false; st = 1; need_load = false; } else run = false;
                } else run = false;
            } else run = false;                                             // Y1: F = Dy F, H = Dy' H;  Y2: H = Dy' H
            if (store) {
                store_nat(v, cur, contig);
                release(curb, true);
                if (contig) release(bB, false);
                if (kind == PH_T && st == 1) { cur = pC; curb = bC; tab = tabd + N; st = 2; need_load = true; }      // next: the stash -> H
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&b_iempty[slot]);
    }
}

}  // namespace fts
#endif
