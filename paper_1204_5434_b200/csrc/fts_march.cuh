// fts_march.cuh — the contour march as ONE persistent kernel per propagator solve.
//
// One RQM4 step (Eq. 12) of a propagator is split into four kinds of work items, each a fused
// 1-D pass over a tile of pencils held in registers (fts_pencil.h):
//
//   T  (x pencils)  finish step s-1:  q_s = (4 e4 Dx'[H] - F)/3  -> slice store;   start step s:  F = Dx[e2 q_s], H = Dx'[e4 q_s]
//   Y1 (y pencils)  F = Dy F,  H = Dy' H
//   Z  (z pencils)  F = e2 Dz F,  H = Dz'[e2 Dz' H]
//   Y2 (y pencils)  H = Dy' H
//
// (D = exp(ds d^2/dx_d^2) applied as FFT -> real table -> IFFT along one dimension, D' the same at ds/2; the three
// 1-D factors of exp(-k^2 ds) commute, so the half branch is ordered x y z | z y x and its two z diffusions meet
// around the real-space multiply.)  F and H are updated in place.  Per step and propagator the items move
// 6 (T) + 4 (Y1) + 5 (Z) + 2 (Y2) fields through L2.  Y1, Z and Y2 can be issued slab by slab over x-ranges small
// enough that a slab of F and H stays resident in the 126 MB L2 from its Y1 read to its Y2 write (HBM then sees
// about 11-13 field transfers per step instead of 17); the default is one slab, because the march is not HBM-bound
// and coarser phases measure faster.
//
// Scheduling: work items are handed out in a fixed global order through an atomic ticket, drawn by one scheduler warp
// per CTA; an item is released to the compute warps (mbarrier ring) when the completion counter of the phase it
// depends on is full.  That phase always precedes it in ticket order, so the kernel is deadlock-free for any grid
// size.  The q and q+ marches are independent; their phases alternate and run half a step apart so that every
// dependency is separated by work of the other propagator.  Data crosses CTAs only through L2: every field access is
// ld.global.cg / st.global.cg / cp.async.
#ifndef FTS_MARCH_CUH
#define FTS_MARCH_CUH

#include <cuda_runtime.h>
#include <stdint.h>

#include "fts_pencil.h"

namespace fts {

enum { PH_T = 0, PH_Y1 = 1, PH_Z = 2, PH_Y2 = 3 };
enum { MARCH_MAXPH = 512, MARCH_SEG_SMEM = 1024 };

struct Phase {              // one entry of the round template ("round" j holds the phases listed in make_template)
    int first;              // first ticket of the phase inside the round
    short chunk;            // x-slab index (Y1, Z, Y2)
    signed char kind;       // PH_*
    signed char prop_off;   // bit 0: propagator b; bit 1: the phase belongs to step (round - 1)
};

// Slice store and density accumulation, shared by both march kernels.  Slices s <= keep and the last slice of the march
// are retained (slot s, resp. keep + 1); store_both keeps every slice (keep = Ns).  With h = Ns/2 the T item that emits
//   q_j   (j > h)   adds  c_j     q_j  q+_{Ns-j}  (stored, Ns-j < h)   into acc[0][species],
//   q+_m  (m >= h)  adds  c_{Ns-m} q+_m q_{Ns-m}  (stored, Ns-m <= h)  into acc[1][species],
// so every pair (j, Ns-j) is visited exactly once and the product is never written.  One propagator (q+ = q): the item of
// q_j, j >= h, adds (c_j + c_{Ns-j}) q_j q_{Ns-j} for j > h and c_h q_h^2 for j = h.  acc is zeroed before the march;
// phi = (ds/Q) (acc[0] + acc[1]) is formed afterwards (density_finish_kernel).
struct DensArgs {
    void* acc[2][2];            // [propagator][species], un-normalised sums; element type = the field type
    const double* cA; const double* cB;     // Simpson weights per contour index (0 outside the block)
    int on;                     // accumulate (full marches only)
    int keep;                   // slices 0..keep are retained at slot s; the last slice of the march at slot keep + 1
    int half;                   // h = Ns / 2
};
__host__ __device__ inline int slice_slot(int s, int keep) { return s <= keep ? s : keep + 1; }

// N1, real-field fast path (the SCFT fields are real).  With real w_A, w_B the propagators
// q and q+ are real, and because every diffusion factor F^-1 exp(-k^2 ds) F is a REAL linear operator, the two marches can
// share one complex march of z = q + i q+:  the Boltzmann multiplies act component-wise, (Re z e_q, Im z e_q+), with the
// factor field packed as (exp(-w_{alpha(s)} ds/4), exp(-w_{alpha+(s)} ds/4)) for the species pair of step s.  Half the
// transforms, half the slices.  species_index() names the factor field of a step; cmul() is the multiply of either mode.
// seg[j] = species of the contour segment [j, j+1] (linear multiblock chains; default: the AB diblock).
// Step s of q crosses segment s; step m of q+ (indexed from the far end, reading A-2) crosses segment Ns - 1 - m.
__device__ __forceinline__ int species_index(int packed, int nspecies, const signed char* seg, int Ns, int b, int step) {
    if (nspecies != 2) return 0;
    step = step < 0 ? 0 : (step > Ns - 1 ? Ns - 1 : step);
    const int sq = seg[step], sqd = seg[Ns - 1 - step];                     // O5 / O6 block schedule of q and of q+
    if (packed) return 2 * sq + sqd;
    return b == 0 ? sq : sqd;
}
template <class T> __device__ __forceinline__ cplx<T> cmul(cplx<T> a, cplx<T> e, bool componentwise) {
    return componentwise ? mk<T>(a.x * e.x, a.y * e.y) : a * e;
}

struct MarchArgs {
    void* q[2]; void* F[2]; void* H[2];
    const void* e4[4];          // Boltzmann factors exp(-w ds/4) per species; packed mode: per (species of q, species of q+) pair
    const void* tab[3][2];      // per dimension: exp(-k_d^2 ds)/N_d, exp(-k_d^2 ds/2)/N_d
    const void* tw[3];          // per dimension: inter-stage twiddles, per-(register, thread) layout
    int g[3];
    long long M;
    int Ns, jA, nspecies, nsteps;
    const signed char* seg;     // species per contour segment (species_index)
    int nprop;                  // propagators marched (2 = diblock q and q+; 1 otherwise, and in packed mode)
    int packed;                 // N1 real-field fast path: ONE complex march of z = q + i q+ (see cmul_mode)
    int nchunks, planes;        // x-slabs and planes per slab
    const Phase* phases; int nphases; int tickets_per_round; int round0, round1;   // rounds [round0, round1]
    int ntT, nY1, nZ, nY2;      // tickets of one T phase / of one slab's Y1, Z, Y2 phase
    unsigned* ticket;           // NULL: one item per CTA (ticket = blockIdx.x) and no dependency waits (stream order)
    unsigned* done;             // completion counters [prop][step][2 + 2*nchunks]: T, Y2 (all slabs), Y1[slab], Z[slab]
    int* err;                   // set to 1 if a dependency wait timed out
    // S6 (Eq. 8): Simpson density sums accumulated by the T items, meet-in-the-middle
    DensArgs dens;
};

template <class T> struct vec2;
template <> struct vec2<double> { typedef double2 type; };
template <> struct vec2<float> { typedef float2 type; };

template <class T> __device__ __forceinline__ cplx<T> ldcg(const cplx<T>* p) {
    typename vec2<T>::type v = __ldcg(reinterpret_cast<const typename vec2<T>::type*>(p));
    return mk<T>(v.x, v.y);
}
template <class T> __device__ __forceinline__ void stcg(cplx<T>* p, cplx<T> v) {
    typename vec2<T>::type w; w.x = v.x; w.y = v.y;
    __stcg(reinterpret_cast<typename vec2<T>::type*>(p), w);
}
// Polling uses relaxed loads; the acquire fence (which invalidates L1) is paid once, when the counter is complete.
__device__ __forceinline__ unsigned ld_relaxed(const unsigned* p) {
    unsigned v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void fence_acquire() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
__device__ __forceinline__ unsigned long long globaltimer_ns() { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }

template <class T, int N, int EPT, int TZ>
struct MarchCfg {
    typedef PencilShape<N, EPT> S;
    static constexpr int TARGET = 128;
    static constexpr int GROUP_S = TZ * S::TPP;                                       // threads of one strided tile [N][TZ]
    static constexpr int GPB_S = (TARGET / GROUP_S) > 0 ? (TARGET / GROUP_S) : 1;     // strided tiles per item
    static constexpr int THREADS = GROUP_S * GPB_S;
    static constexpr int GPB_C = THREADS / S::TPP;                                    // contiguous pencils per item
    static constexpr int PS = contig_ps<T, N, EPT>();
    static constexpr int XELEMS = S::ONE ? 1 : ((GPB_C * PS > GPB_S * N * TZ) ? GPB_C * PS : GPB_S * N * TZ);
    typedef XchgLayout<PS, S::R2 + 1, 1> LC;
    typedef XchgLayout<1, S::R2 * TZ, TZ> LS;
    static constexpr size_t SMEM = (size_t)N * sizeof(cplx<T>) + 2 * (size_t)N * sizeof(T) + (size_t)XELEMS * sizeof(cplx<T>) +
                                   2 * (size_t)THREADS * EPT * sizeof(cplx<T>) + (size_t)MARCH_MAXPH * sizeof(Phase);
    static constexpr int LAUNCH = THREADS + 32;                                       // + one scheduler warp
    static constexpr int MINB = (sizeof(T) == 8 && EPT == 16) ? 2 : ((THREADS <= 128) ? 3 : 2);
};

// barrier among the NT compute threads of a CTA (the scheduler warp does not take part)
template <int NT, int ID = 1> __device__ __forceinline__ void bar_compute() { asm volatile("bar.sync %0, %1;" ::"n"(ID), "n"(NT) : "memory"); }

// mbarrier primitives (shared memory, CTA scope): the scheduler warp and the compute warps hand items back and forth
__device__ __forceinline__ void mbar_init(uint64_t* b, unsigned count) {
    asm volatile("mbarrier.init.shared.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* b) {
    asm volatile("{ .reg .b64 st; mbarrier.arrive.shared.b64 st, [%0]; }" ::"r"((unsigned)__cvta_generic_to_shared(b)) : "memory");
}
__device__ __forceinline__ bool mbar_test(uint64_t* b, unsigned parity) {
    unsigned ok;
    asm volatile("{ .reg .pred p; mbarrier.test_wait.parity.shared.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                 : "=r"(ok) : "r"((unsigned)__cvta_generic_to_shared(b)), "r"(parity) : "memory");
    return ok != 0;
}
// A wait inside a CTA (descriptor hand-off) can only fail through a bug: it traps after 20 s of wall clock (the launch then
// fails loudly with a CUDA error) instead of hanging the GPU or leaving a barrier half-arrived.
__device__ __forceinline__ bool mbar_wait(uint64_t* b, unsigned parity) {
    unsigned ok, tries = 0;
    unsigned long long t0 = 0;
    for (;;) {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                     : "=r"(ok) : "r"((unsigned)__cvta_generic_to_shared(b)), "r"(parity) : "memory");
        if (ok) return true;
        if ((++tries & 4095u) == 0) {
            unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
            if (t0 == 0) t0 = t; else if (t - t0 > 20000000000ull) __trap();
        }
    }
}

// exp(a ds d^2/dx_d^2) along the pencil: forward transform, real table (1/N folded in), inverse transform.
// One shared-memory buffer serves both exchanges: every thread overwrites only what it last read.  `contig`
// (block-uniform) selects the exchange addressing of the z pass (LC) or of the x/y passes (LS); the butterflies are shared.
template <class T, int N, int EPT, int NT, class LS, class LC, int BAR = 1>
__device__ __forceinline__ void diffuse(cplx<T> (&v)[EPT], int t, int p, bool contig, const cplx<T>* s_tw, const T* tab, cplx<T>* xs, cplx<T>* xc) {
    typedef Pencil<T, N, EPT> P;
    typedef PencilShape<N, EPT> S;
    P::fwd_a(v, t, s_tw);
    if constexpr (!S::ONE) {
        if (contig) P::template xchg_store_a<LC>(v, t, xc, p); else P::template xchg_store_a<LS>(v, t, xs, p);
        bar_compute<NT, BAR>();
        if (contig) P::template xchg_load_b<LC>(v, t, xc, p); else P::template xchg_load_b<LS>(v, t, xs, p);
    }
    P::fwd_b(v);
#pragma unroll
    for (int r = 0; r < EPT; ++r) v[r] = v[r] * tab[t + S::TPP * r];
    P::inv_b(v);
    if constexpr (!S::ONE) {
        if (contig) P::template xchg_store_b<LC>(v, t, xc, p); else P::template xchg_store_b<LS>(v, t, xs, p);
        bar_compute<NT, BAR>();
        if (contig) P::template xchg_load_a<LC>(v, t, xc, p); else P::template xchg_load_a<LS>(v, t, xs, p);
    }
    P::inv_a(v, t, s_tw);
}

// cp.async of one complex element (generic proxy, so ordinary acquire/release ordering applies): 16 bytes bypass L1;
// 8 bytes (complex64) go through L1, which the dependency acquire of the item has invalidated.
template <class T> __device__ __forceinline__ void cp_async_elem(cplx<T>* smem_dst, const cplx<T>* gsrc) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
    if constexpr (sizeof(T) == 8) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gsrc) : "memory");
    else asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sa), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int NLEFT> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(NLEFT) : "memory"); }

// Coordinates of one thread inside a work item.  Recomputed from the item descriptor in shared memory wherever they are
// needed (a few integer instructions) instead of being kept live across the transforms, where they would spill.
template <class T>
struct Coords {
    int kind, job, s, b, chunk;
    bool active;
    int base0, estride;                     // element offset of register r inside a field: base0 + r*estride   (M <= 2^24)
};

enum { MARCH_RING = 4, MARCH_RING_F32 = 2 };      // item descriptors in flight between the scheduler warp and the compute warps
                                                   // (A/B: complex64 with its 3 CTAs/SM balances better with fewer tickets held per CTA)

template <class T, int N, int EPT, int TZ>
__global__ void __launch_bounds__(MarchCfg<T, N, EPT, TZ>::LAUNCH, MarchCfg<T, N, EPT, TZ>::MINB) march_kernel(const MarchArgs A) {
    typedef MarchCfg<T, N, EPT, TZ> Cfg;
    typedef typename Cfg::S S;
    typedef typename Cfg::LS LS;
    typedef typename Cfg::LC LC;
    typedef cplx<T> C;
    constexpr int TPP = S::TPP;
    constexpr int NT = Cfg::THREADS;          // compute threads; warp NT/32 is the scheduler
    constexpr int R = sizeof(T) == 4 ? MARCH_RING_F32 : MARCH_RING;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* s_tw = reinterpret_cast<C*>(smem_raw);
    T* s_tab = reinterpret_cast<T*>(s_tw + N);
    C* s_x = reinterpret_cast<C*>(s_tab + 2 * N);          // exchange buffer of the transforms
    C* s_stash = s_x + Cfg::XELEMS;                        // thread-private [r][tid]: e4 tile, then the stashed half-branch input
    C* s_pre = s_stash + NT * EPT;                         // thread-private [r][tid]: primary input of the NEXT item (and F of a T item)
    Phase* s_ph = reinterpret_cast<Phase*>(s_pre + NT * EPT);
    __shared__ signed char s_seg[MARCH_SEG_SMEM];      // species per contour segment (a global load per lookup would sit on every item's critical path)
    __shared__ int s_item[R][4];              // step, phase index, index inside the phase, state (0: end of march, 1: work)
    __shared__ __align__(8) uint64_t s_full[R], s_done[R];

    const int tid = threadIdx.x;
    for (int i = tid; i < A.nphases; i += Cfg::LAUNCH) s_ph[i] = A.phases[i];
    const bool seg_in_smem = A.Ns <= MARCH_SEG_SMEM;
    if (seg_in_smem && A.nspecies == 2) for (int i = tid; i < A.Ns; i += Cfg::LAUNCH) s_seg[i] = A.seg[i];
    const signed char* const seg = seg_in_smem ? s_seg : A.seg;
    if (tid == 0) {
        for (int i = 0; i < R; ++i) { mbar_init(&s_full[i], 1); mbar_init(&s_done[i], NT); }
    }
    const int C2 = 2 + 2 * A.nchunks;         // counters per (propagator, step)
    const unsigned total = (unsigned)((A.round1 - A.round0 + 1) * A.tickets_per_round);
    __syncthreads();
    // Per-phase launch mode chains ~4 Ns tiny kernels: with programmatic dependent launch the next kernel's CTAs are scheduled
    // and run the prologue above (constant tables only) while this one's last stores drain (the trigger is at the END of a
    // CTA's work: triggered at the start, the waiting CTAs of the next phase crowd the SMs and a 32^3 march gets 20 % slower);
    // everything below reads what the previous kernel wrote and therefore waits for its completion and memory flush here.
    // (No-ops without the launch attribute.)
    asm volatile("griddepcontrol.wait;" ::: "memory");

    if (tid >= NT) {
        // ================= scheduler warp: one thread draws tickets, resolves dependencies, signals completions =================
        if (tid != NT) return;
        // the completion counter an item of (phase, step) waits for, and the count it needs
        auto dependency = [&](const Phase& ph, int s, unsigned& need) -> const unsigned* {
            const int b = ph.prop_off & 1;
            const unsigned* cnt = A.done + ((size_t)b * (A.Ns + 1) + s) * C2;
            need = 0;
            if (ph.kind == PH_T) { if (s <= 0) return nullptr; need = (unsigned)(A.nchunks * A.nY2); return cnt - C2 + 1; }
            if (ph.kind == PH_Y1) { need = (unsigned)A.ntT; return cnt; }
            if (ph.kind == PH_Z) { need = (unsigned)A.nY1; return cnt + 2 + ph.chunk; }
            need = (unsigned)A.nZ; return cnt + 2 + A.nchunks + ph.chunk;
        };
        // T items that accumulate densities also read a slice the OTHER propagator (or, with one propagator, an earlier step)
        // stored: its T phase must be complete.  It lies at least a step back in ticket order, so this never waits in practice.
        auto dependency2 = [&](const Phase& ph, int s, unsigned& need) -> const unsigned* {
            need = 0;
            if (ph.kind != PH_T || !A.dens.on) return nullptr;
            const int b = ph.prop_off & 1, nprop = A.nprop;
            if (nprop == 2 ? (b == 0 ? s <= A.dens.half : s < A.dens.half) : s <= A.dens.half) return nullptr;
            need = (unsigned)A.ntT;
            return A.done + ((size_t)(nprop == 2 ? 1 - b : 0) * (A.Ns + 1) + (A.Ns - s)) * C2;
        };
        unsigned issued = 0, completed = 0;
        unsigned long long t_wait0 = 0; unsigned spins = 0;
        bool aborted = false;
        const unsigned* pw2 = nullptr; unsigned pneed2 = 0;
        unsigned tk_pending = A.ticket ? atomicAdd(A.ticket, 1u) : blockIdx.x;       // drawn one item ahead
        bool have = false, exhausted = false;
        int ps = 0, plo = 0, pidx = 0;                 // the item waiting for its dependency
        const unsigned* pw = nullptr; unsigned pneed = 0;
        const unsigned* dep_ok = nullptr;              // a counter once seen complete stays complete
        int lo = 0;
        for (;;) {
            bool progress = false;
            if (completed < issued) {                  // oldest item in flight: have all compute threads issued its stores?
                const int slot = completed % R;
                if (mbar_test(&s_done[slot], (completed / R) & 1)) {
                    if (A.ticket) {
                        const Phase ph = s_ph[s_item[slot][1]];
                        const int b = ph.prop_off & 1, s = s_item[slot][0];
                        unsigned* cnt = A.done + ((size_t)b * (A.Ns + 1) + s) * C2;
                        unsigned* c = ph.kind == PH_T ? cnt : ph.kind == PH_Y2 ? cnt + 1 : ph.kind == PH_Y1 ? cnt + 2 + ph.chunk : cnt + 2 + A.nchunks + ph.chunk;
                        __threadfence();
                        atomicAdd(c, 1u);
                    }
                    ++completed; progress = true;
                }
            }
            if (!exhausted && issued - completed < (unsigned)R) {
                if (!have) {
                    const unsigned tk = tk_pending;
                    if (tk >= total) {                 // end of march: publish the sentinel
                        const int slot = issued % R;
                        s_item[slot][3] = 0;
                        mbar_arrive(&s_full[slot]);
                        exhausted = true;
                        continue;
                    }
                    tk_pending = A.ticket ? atomicAdd(A.ticket, 1u) : total;
                    const int round = A.round0 + (int)(tk / (unsigned)A.tickets_per_round), off = (int)(tk % (unsigned)A.tickets_per_round);
                    if (s_ph[lo].first > off) lo = 0;                                  // new round: restart the phase scan
                    while (lo + 1 < A.nphases && s_ph[lo + 1].first <= off) ++lo;
                    const Phase ph = s_ph[lo];
                    ps = round - ((ph.prop_off >> 1) & 1); plo = lo; pidx = off - ph.first;
                    const bool live = ph.kind == PH_T ? (ps >= 0 && ps <= A.nsteps) : (ps >= 0 && ps < A.nsteps);
                    if (!live) continue;               // ticket of a phase outside the march: no work
                    pw = A.ticket ? dependency(ph, ps, pneed) : nullptr;
                    pw2 = A.ticket ? dependency2(ph, ps, pneed2) : nullptr;
                    have = true; spins = 0; t_wait0 = 0;
                }
                bool ok = (!pw || pw == dep_ok) && !pw2;
                if (!ok) {
                    ok = (!pw || pw == dep_ok || ld_relaxed(pw) >= pneed) && (!pw2 || ld_relaxed(pw2) >= pneed2);
                    if (!ok && (++spins & 1023u) == 0) {
                        // another CTA's work is 5 s late (wall clock): a bug or a lost CTA.  Flag it and DRAIN: no further item is
                        // released, the compute warps get the end sentinel, Q is poisoned by the reduction (never compute on).
                        const unsigned long long now = globaltimer_ns();
                        if (t_wait0 == 0) t_wait0 = now;
                        else if (now - t_wait0 > 5000000000ull) { atomicExch(A.err, 1); aborted = true; }
                    }
                    if (ok) fence_acquire();
                }
                if (aborted) {
                    const int slot = issued % R;
                    s_item[slot][3] = 0;
                    mbar_arrive(&s_full[slot]);
                    exhausted = true; have = false;
                    continue;
                }
                if (ok) {
                    if (pw) dep_ok = pw;
                    const int slot = issued % R;
                    s_item[slot][0] = ps; s_item[slot][1] = plo; s_item[slot][2] = pidx; s_item[slot][3] = 1;
                    mbar_arrive(&s_full[slot]);
                    ++issued; have = false; progress = true;
                }
            }
            if (exhausted && completed == issued) break;
            if (!progress) __nanosleep(32);
        }
        return;
    }

    // ================= compute warps =================
    // every thread: its coordinates inside the item published in s_item[slot]
    const int Ny = A.g[1], Nz = A.g[2];
    auto coords = [&](int slot, Coords<T>& c) {
        const volatile int* it = s_item[slot];
        c.s = it[0];
        const Phase ph = s_ph[it[1]];
        const int idx = it[2];
        c.b = ph.prop_off & 1; c.kind = ph.kind; c.chunk = ph.chunk; c.job = 0;
        if (c.kind == PH_Z) {                                         // GPB_C pencils per item, lanes run along the pencil
            const int per_job = A.nZ >> 1;
            c.job = idx >= per_job;
            const int local = (idx - c.job * per_job) * Cfg::GPB_C + tid / TPP;
            c.active = local < A.planes * Ny;
            c.base0 = (c.chunk * A.planes * Ny + local) * N + tid % TPP;
            c.estride = TPP;
        } else {                                                      // tiles [N][TZ], lanes run along z (the contiguous direction)
            const int zz = tid % TZ, tb = tid / (TZ * TPP), t = (tid / TZ) % TPP;
            if (c.kind == PH_T) {
                const int tile = idx * Cfg::GPB_S + tb;
                c.active = tile < (Ny * Nz) / TZ;
                c.base0 = tile * TZ + zz + t * (Ny * Nz);
                c.estride = Ny * Nz * TPP;
            } else {
                const int tpp_z = Nz / TZ, lg = 31 - __clz(tpp_z);    // tiles per plane (a power of two)
                int tg = idx;
                c.job = 1;
                if (c.kind == PH_Y1) { const int per_job = A.nY1 >> 1; c.job = idx >= per_job; tg = idx - c.job * per_job; }
                const int local = tg * Cfg::GPB_S + tb;
                c.active = local < A.planes * tpp_z;
                const int tile = c.chunk * A.planes * tpp_z + local;
                c.base0 = (tile >> lg) * Ny * Nz + (tile & (tpp_z - 1)) * TZ + zz + t * Nz;
                c.estride = Nz * TPP;
            }
        }
    };
    auto primary_src = [&](const Coords<T>& c) { return static_cast<const C*>((c.kind == PH_T || c.job == 1) ? A.H[c.b] : A.F[c.b]); };
    auto prefetch_tile = [&](C* dst, const C* src, const Coords<T>& c) {      // this thread's EPT points -> dst[r][tid]
        if (c.active) {
#pragma unroll
            for (int r = 0; r < EPT; ++r) cp_async_elem<T>(dst + r * NT + tid, src + c.base0 + r * c.estride);
        }
        cp_async_commit();
    };
    // species of contour step `step` of propagator b (O5 / O6 block schedule)
    auto species = [&](int b, int step) -> int { return species_index(A.packed, A.nspecies, seg, A.Ns, b, step); };
    const bool cw = A.packed != 0;

    int cur_dim = -1;
    bool cur_pref = false;
    for (unsigned it = 0;; ++it) {
        const int slot = it % R, nslot = (it + 1) % R;
        if (!mbar_wait(&s_full[slot], (it / R) & 1)) { atomicExch(A.err, 1); break; }      // descriptor published, dependency met
        if (((const volatile int*)s_item[slot])[3] == 0) break;
        bool nxt_pref = false;
        // stage the next item's primary input into s_pre if the scheduler has already released it (per-thread decision:
        // the staging buffers are thread-private)
        auto stage_next = [&]() {
            if (mbar_test(&s_full[nslot], ((it + 1) / R) & 1) && ((const volatile int*)s_item[nslot])[3] == 1) {
                Coords<T> n; coords(nslot, n);
                if (!(n.kind == PH_T && n.s == 0)) { prefetch_tile(s_pre, primary_src(n), n); nxt_pref = true; }
            }
        };

        C v[EPT];
        int kind, st = 0, job = 0;
        bool contig;
        {   // ---- load phase ----
            Coords<T> c; coords(slot, c);
            kind = c.kind; contig = kind == PH_Z; job = c.job;
            const int dim = kind == PH_T ? 0 : (kind == PH_Z ? 2 : 1);
            if (dim != cur_dim) {                      // new tables, possibly a new exchange layout: everyone must be done with the old
                bar_compute<NT>();
                for (int i = tid; i < N; i += NT) {
                    s_tw[i] = static_cast<const C*>(A.tw[dim])[i];
                    s_tab[i] = static_cast<const T*>(A.tab[dim][0])[i];
                    s_tab[N + i] = static_cast<const T*>(A.tab[dim][1])[i];
                }
                cur_dim = dim;
                bar_compute<NT>();
            }
            const bool finish = c.s > 0;
            // secondary input e4 -> s_stash, needed after the first diffusion (T finish, Z)
            const bool e4_staged = (kind == PH_T && finish) || kind == PH_Z;
            if (e4_staged) prefetch_tile(s_stash, static_cast<const C*>(A.e4[species(c.b, kind == PH_T ? c.s - 1 : c.s)]), c);
            if (!(kind == PH_T && !finish)) {                         // primary input: staged by the previous iteration, or loaded directly
                if (cur_pref) {
                    if (e4_staged) cp_async_wait<1>(); else cp_async_wait<0>();
#pragma unroll
                    for (int r = 0; r < EPT; ++r) v[r] = s_pre[r * NT + tid];
                } else {
                    const C* src = primary_src(c);
#pragma unroll
                    for (int r = 0; r < EPT; ++r) v[r] = c.active ? ldcg(src + c.base0 + r * c.estride) : mk<T>(0, 0);
                }
            }
            // s_pre is free again: T items stage F for the combine, the others stage the next item's primary input now
            if (kind == PH_T) { if (finish) prefetch_tile(s_pre, static_cast<const C*>(A.F[c.b]), c); }
            else stage_next();
        }
        // T item tail: from q_s in v, write the slice, then b = e4 q_s -> stash, a = e4 b -> v   (start of step s)
        auto emit_q_and_start = [&](bool combine) {
            Coords<T> c; coords(slot, c);
            const bool start = c.s < A.nsteps;
            const int sp_now = species(c.b, c.s), sp_prev = species(c.b, c.s - 1);
            const bool keep = c.s <= A.dens.keep || c.s == A.nsteps;
            C* qs = static_cast<C*>(A.q[c.b]) + (long long)slice_slot(c.s, A.dens.keep) * A.M;
            // density pair of this slice (DensArgs): partner slice and Simpson weights
            const bool two = A.nprop == 2;
            const int h = A.dens.half, jp = (two && c.b == 1) ? A.Ns - c.s : c.s;      // contour index j of the pair (j, Ns - j)
            const bool dens = A.dens.on && (two ? (c.b == 0 ? c.s > h : c.s >= h) : c.s >= h);
            const bool self = !two && c.s == h;
            const C* partner = static_cast<const C*>(A.q[two ? 1 - c.b : 0]) + (long long)(A.Ns - c.s) * A.M;      // stored: Ns - s <= keep
            double wA = 0.0, wB = 0.0;
            double wA2 = 0.0, wB2 = 0.0;                              // packed mode: the mirror pair (Ns - s, s)
            if (dens) {
                wA = A.dens.cA[jp]; wB = A.dens.cB[jp];
                if (cw) { if (!self) { wA2 = A.dens.cA[A.Ns - jp]; wB2 = A.dens.cB[A.Ns - jp]; } }
                else if (!two && !self) wA += A.dens.cA[A.Ns - jp];
            }
            C* accA = static_cast<C*>(A.dens.acc[c.b][0]); C* accB = static_cast<C*>(A.dens.acc[c.b][1]);
            const C* e4s = static_cast<const C*>(A.e4[sp_now]);
            const bool reload = !combine || sp_now != sp_prev;
#pragma unroll
            for (int r = 0; r < EPT; ++r) {
                const int i = c.base0 + r * c.estride;
                if (combine) {                                        // q_s = (4 e4 Dx'[H] - F)/3     (Eq. 12)
                    const C e = s_stash[r * NT + tid];
                    const C f = s_pre[r * NT + tid];
                    const C h = cmul(v[r], e, cw);
                    v[r] = mk<T>(((T)4 * h.x - f.x) * (T)(1.0 / 3.0), ((T)4 * h.y - f.y) * (T)(1.0 / 3.0));
                }
                if (c.active && keep) stcg(qs + i, v[r]);             // the slice store IS the step's output write
            }
            if (dens && c.active) {
                // Eq. 8: this slice times the stored partner, weighted, into the sums.  All loads of a batch are issued before its
                // first store (the compiler cannot hoist them itself: the stores might alias), so a batch costs ONE round trip.
                constexpr int BATCH = EPT < (sizeof(T) == 8 ? 4 : 8) ? EPT : (sizeof(T) == 8 ? 4 : 8);
                for (int pass = 0; pass < 2; ++pass) {                // species A, then B (both only at the block junction)
                    const double w1 = pass == 0 ? wA : wB;
                    if (cw ? pass == 1 : w1 == 0.0) continue;
                    C* acc = cw ? accA : (pass == 0 ? accA : accB);
#pragma unroll
                    for (int r0 = 0; r0 < EPT; r0 += BATCH) {
                        C zp[BATCH], a[BATCH];
#pragma unroll
                        for (int k = 0; k < BATCH; ++k) {
                            const int i = c.base0 + (r0 + k) * c.estride;
                            zp[k] = self ? v[r0 + k] : ldcg(partner + i);
                            a[k] = ldcg(acc + i);
                        }
#pragma unroll
                        for (int k = 0; k < BATCH; ++k) {
                            const int i = c.base0 + (r0 + k) * c.estride;
                            const C q = v[r0 + k];
                            if (cw) {                                 // z = q + i q+: pairs (s, Ns-s) and (Ns-s, s); sums (A, B) as (re, im)
                                const T p1 = q.x * zp[k].y, p2 = zp[k].x * q.y;
                                stcg(acc + i, mk<T>(a[k].x + (T)wA * p1 + (T)wA2 * p2, a[k].y + (T)wB * p1 + (T)wB2 * p2));
                            } else {
                                const C pr = q * zp[k];
                                stcg(acc + i, mk<T>(a[k].x + (T)w1 * pr.x, a[k].y + (T)w1 * pr.y));
                            }
                        }
                    }
                }
            }
            if (start) {
#pragma unroll
                for (int r = 0; r < EPT; ++r) {
                    const int i = c.base0 + r * c.estride;
                    C e;
                    if (reload) e = c.active ? ldcg(e4s + i) : mk<T>(0, 0);
                    else e = s_stash[r * NT + tid];
                    const C hb = cmul(v[r], e, cw);
                    s_stash[r * NT + tid] = hb;
                    v[r] = cmul(hb, e, cw);
                }
            }
            return start;
        };
        auto store_tile = [&](int which) {                            // 0: F, 1: H of the item's propagator
            Coords<T> c; coords(slot, c);
            C* dst = static_cast<C*>(which ? A.H[c.b] : A.F[c.b]);
            if (c.active) {
#pragma unroll
                for (int r = 0; r < EPT; ++r) stcg(dst + c.base0 + r * c.estride, v[r]);
            }
        };

        bool run = true;
        if (kind == PH_T && ((const volatile int*)s_item[slot])[0] == 0) {      // q(x,0) = 1, q+(x,s=1) = 1
#pragma unroll
            for (int r = 0; r < EPT; ++r) v[r] = mk<T>(1, cw ? 1 : 0);      // packed: z_0 = q_0 + i q+_0 = 1 + i
            run = emit_q_and_start(false);
            stage_next();
            st = 1;
        }
#pragma unroll 1
        while (run) {
            // thread position inside the transform, and the table: full step for the F branch, half step otherwise
            const int t = contig ? tid % TPP : (tid / TZ) % TPP, p = contig ? tid / TPP : tid % TZ;
            C* xs = contig ? s_x : s_x + (tid / (TZ * TPP)) * (N * TZ);
            const bool full = kind == PH_T ? (st == 1) : (job == 0);
            diffuse<T, N, EPT, NT, LS, LC>(v, t, p, contig, s_tw, full ? s_tab : s_tab + N, xs, s_x);
            if (kind == PH_T) {
                if (st == 0) {
                    cp_async_wait<0>();                               // e4 and F tiles of this item
                    run = emit_q_and_start(true);
                    stage_next();
                    st = 1;
                } else if (st == 1) {
                    store_tile(0);
#pragma unroll
                    for (int r = 0; r < EPT; ++r) v[r] = s_stash[r * NT + tid];
                    st = 2;
                } else {
                    store_tile(1);
                    run = false;
                }
            } else if (kind == PH_Z && st == 0) {                     // F = e2 Dz F;  H = Dz'[e2 Dz' H]
                if (nxt_pref) cp_async_wait<1>(); else cp_async_wait<0>();      // the e4 tile (committed before the next item's tile)
#pragma unroll
                for (int r = 0; r < EPT; ++r) {
                    const C e = s_stash[r * NT + tid];
                    v[r] = cmul(v[r], cmul(e, e, cw), cw);
                }
                if (job == 0) { store_tile(0); run = false; }
                st = 1;
            } else {                                                  // Y1, Y2, second z diffusion of H
                store_tile(job);
                run = false;
            }
        }
        mbar_arrive(&s_done[slot]);                                   // this thread's stores of the item are issued
        cur_pref = nxt_pref;
    }
    cp_async_wait<0>();
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

}  // namespace fts
#endif
