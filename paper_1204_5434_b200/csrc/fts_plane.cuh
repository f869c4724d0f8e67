// fts_plane.cuh — the kernels of the per-phase launch mode on small grids: plane_kernel (the y and z diffusions of one RQM4
// step fused per yz-plane, Ny = Nz = 16, 32 or 64) and tline_kernel (the x pencils of a step as a straight-line kernel).
//
// On small grids a contour step is bound by the latency of its phases, not by any pipe: in the per-phase
// launch mode a step is four kernels (T, Y1, Z, Y2) of a few microseconds each.  Y1, Z and Y2 act inside yz-planes
// (fts_march.cuh), and at these sizes the planes a CTA holds in registers (NT * EPT points: eight planes at N = 16 and one at
// N = 32 with 128 threads, one at N = 64 with 512 threads) are exactly the planes its Y items and its Z items cover, so the three phases collapse into ONE
// kernel that passes the planes between the y layout (lanes along z) and the z layout (lanes along the pencil) through
// shared memory:
//
//   job F:  F <- e2 Dz Dy F                          (2 diffusions)
//   job H:  H <- Dy' Dz' [ e2 Dz' Dy' H ]            (4 diffusions)
//
// A step is then two kernels, T (march_kernel) and this one.  Same butterflies, tables and arithmetic order as the Y1 / Z /
// Y2 items, so the results are bit-identical to the other march modes.
#ifndef FTS_PLANE_CUH
#define FTS_PLANE_CUH

#include "fts_march.cuh"

namespace fts {

struct PlaneArgs {
    void* F[2]; void* H[2]; const void* e4[4];
    const void* tab[2][2];      // [y, z][full, half]: exp(-k_d^2 ds)/N_d, exp(-k_d^2 ds/2)/N_d
    const void* tw[2];          // [y, z] inter-stage twiddles
    const signed char* seg;
    int Nx, Ns, nspecies, nprop, packed, step;
};

template <class T, int N, int EPT>
struct PlaneCfg {
    typedef PencilShape<N, EPT> S;
    static constexpr int NT = N == 64 ? 512 : 128, TZ = 8;
    static constexpr int PL = NT * EPT / (N * N);                       // planes per CTA
    static constexpr int GPB_S = NT / (TZ * S::TPP), GPB_C = NT / S::TPP;
    static constexpr int PS = contig_ps<T, N, EPT>();
    static constexpr int XELEMS = S::ONE ? 1 : ((GPB_C * PS > GPB_S * N * TZ) ? GPB_C * PS : GPB_S * N * TZ);
    // plane rows are padded so that both layouts are conflict-free for complex128 (y layout: 128-byte row segments; z layout:
    // TPP consecutive elements of 8 / TPP rows per wavefront)
    static constexpr int ROW = N + (S::ONE ? 1 : 4);
    typedef XchgLayout<PS, S::R2 + 1, 1> LC;
    typedef XchgLayout<1, S::R2 * TZ, TZ> LS;
    static constexpr size_t SMEM = (size_t)(2 * N + XELEMS + PL * N * ROW) * sizeof(cplx<T>) + 4 * (size_t)N * sizeof(T);
    static_assert(PL >= 1 && PL * N * N == NT * EPT && GPB_S * TZ == PL * N && GPB_C == PL * N, "a CTA must hold whole planes in both layouts");
};

template <class T, int N, int EPT>
__global__ void __launch_bounds__(PlaneCfg<T, N, EPT>::NT) plane_kernel(const PlaneArgs A) {
    typedef PlaneCfg<T, N, EPT> Cfg;
    typedef typename Cfg::S S;
    typedef cplx<T> C;
    constexpr int TPP = S::TPP, NT = Cfg::NT, TZ = Cfg::TZ, ROW = Cfg::ROW;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* s_tw = reinterpret_cast<C*>(smem_raw);                  // [y, z][N]
    T* s_tab = reinterpret_cast<T*>(s_tw + 2 * N);             // [y, z][full, half][N]
    C* s_x = reinterpret_cast<C*>(s_tab + 4 * N);              // exchange buffer of the transforms
    C* s_pl = s_x + Cfg::XELEMS;                               // the CTA's planes, [plane][y][ROW]

    const int tid = threadIdx.x;
    for (int i = tid; i < 2 * N; i += NT) s_tw[i] = static_cast<const C*>(A.tw[i / N])[i % N];
    for (int i = tid; i < 4 * N; i += NT) s_tab[i] = static_cast<const T*>(A.tab[i / (2 * N)][(i / N) & 1])[i % N];
    // blockIdx.x -> (propagator, job, plane group)
    const int groups = A.Nx / Cfg::PL;
    const int grp = blockIdx.x % groups, job = (blockIdx.x / groups) & 1, b = blockIdx.x / (2 * groups);
    const int sp = species_index(A.packed, A.nspecies, A.seg, A.Ns, b, A.step);
    const bool cw = A.packed != 0;
    __syncthreads();
    asm volatile("griddepcontrol.wait;" ::: "memory");         // see march_kernel: everything below reads the previous kernel's output

    C* field = static_cast<C*>(job ? A.H[b] : A.F[b]) + (size_t)grp * Cfg::PL * N * N;
    const C* e4 = static_cast<const C*>(A.e4[sp]) + (size_t)grp * Cfg::PL * N * N;
    // y layout: tiles [N y][8 z], lanes along z;  z layout: pencil p = (plane, y), lanes along the pencil
    const int zz = tid % TZ, tb = tid / (TZ * TPP), ty = (tid / TZ) % TPP;
    const int ypl = tb / (N / TZ), yz = (tb % (N / TZ)) * TZ + zz;              // plane and z of this thread's y pencil
    const int tz = tid % TPP, zp = tid / TPP;                                   // z layout: zp = plane * N + y
    C* xs = s_x + tb * (N * TZ);
    const T* taby = s_tab + (job ? N : 0);                                      // full step for F, half step for H
    const T* tabz = s_tab + 2 * N + (job ? N : 0);

    C v[EPT];
#pragma unroll
    for (int r = 0; r < EPT; ++r) v[r] = ldcg(field + ((size_t)ypl * N + (ty + TPP * r)) * N + yz);
    diffuse<T, N, EPT, NT, typename Cfg::LS, typename Cfg::LC>(v, ty, zz, false, s_tw, taby, xs, s_x);
#pragma unroll
    for (int r = 0; r < EPT; ++r) s_pl[(ypl * N + ty + TPP * r) * ROW + yz] = v[r];
    __syncthreads();
#pragma unroll
    for (int r = 0; r < EPT; ++r) v[r] = s_pl[zp * ROW + tz + TPP * r];
    diffuse<T, N, EPT, NT, typename Cfg::LS, typename Cfg::LC>(v, tz, zp, true, s_tw + N, tabz, xs, s_x);
#pragma unroll
    for (int r = 0; r < EPT; ++r) { const C e = ldcg(e4 + (size_t)zp * N + tz + TPP * r); v[r] = cmul(v[r], cmul(e, e, cw), cw); }
    if (job == 0) {                                            // F = e2 Dz Dy F
#pragma unroll
        for (int r = 0; r < EPT; ++r) stcg(field + (size_t)zp * N + tz + TPP * r, v[r]);
    } else {                                                   // H = Dy' Dz' [e2 Dz' Dy' H]
        diffuse<T, N, EPT, NT, typename Cfg::LS, typename Cfg::LC>(v, tz, zp, true, s_tw + N, tabz, xs, s_x);
        __syncthreads();                                       // every thread has read its z pencil before the planes are overwritten
#pragma unroll
        for (int r = 0; r < EPT; ++r) s_pl[zp * ROW + tz + TPP * r] = v[r];
        __syncthreads();
#pragma unroll
        for (int r = 0; r < EPT; ++r) v[r] = s_pl[(ypl * N + ty + TPP * r) * ROW + yz];
        diffuse<T, N, EPT, NT, typename Cfg::LS, typename Cfg::LC>(v, ty, zz, false, s_tw, taby, xs, s_x);
#pragma unroll
        for (int r = 0; r < EPT; ++r) stcg(field + ((size_t)ypl * N + (ty + TPP * r)) * N + yz, v[r]);
    }
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

// ------------------------------------------------------------------------------------------------
// tline_kernel: the T item (x pencils) of one step as a straight-line kernel for the per-phase launch mode.
//
//   q_s = (4 e4 Dx'[H] - F)/3  -> slice store (if retained) and density sums (DensArgs);   F = Dx[e2 q_s],  H = Dx'[e4 q_s]
//
// march_kernel serves the same item through its scheduler warp, descriptor ring and staging buffers - machinery a kernel
// that processes exactly one item per CTA does not need; on small grids, where a step is a chain of two few-microsecond
// kernels, that overhead is a third of the T kernel.  Same butterflies, tables and arithmetic order: bit-identical results.
// One CTA = GPB_S tiles [N x][8 z]; blockIdx.x -> (propagator, tile group).  SPLIT: a second group of 128 threads takes the
// half branch (it receives e4 q_s through shared memory and runs Dx' while the first group runs Dx on e2 q_s), so the item's
// critical path is two diffusions instead of three.  The per-phase launch at the middle of the chain is split per
// propagator by the host (q+'s item reads the slice q's item of the same step stores).
// ------------------------------------------------------------------------------------------------
struct TlineArgs {
    void* q[2]; void* F[2]; void* H[2]; const void* e4[4];
    const void* tab[2];         // x dimension: exp(-k_x^2 ds)/Nx, exp(-k_x^2 ds/2)/Nx
    const void* tw;
    const signed char* seg;
    long long M;                // points per field
    int plane;                  // Ny * Nz: element stride along x
    int Ns, nspecies, nprop, packed, step, nsteps;
    int b0, nb;                 // propagators b0 .. b0 + nb - 1
    DensArgs dens;
};

template <class T, int N, int EPT>
struct TlineCfg {
    typedef PencilShape<N, EPT> S;
    static constexpr int NT = 128, TZ = 8;
    static constexpr int GPB_S = NT / (TZ * S::TPP);
    static constexpr int XELEMS = S::ONE ? 1 : GPB_S * N * TZ;
    typedef XchgLayout<1, S::R2 * TZ, TZ> LS;
    typedef XchgLayout<1, S::R2 + 1, 1> LC;                 // unused (strided layout only)
    static constexpr bool SPLIT = N == 64;                   // measured: 64^3 one propagator 2.13 -> 1.93 ms; no gain at 32, a loss at 16 (ONE-thread pencils)
    static constexpr int LAUNCH = SPLIT ? 2 * NT : NT;
    static constexpr size_t SMEM = (size_t)(N + (SPLIT ? 2 : 1) * XELEMS + NT * EPT) * sizeof(cplx<T>) + 2 * (size_t)N * sizeof(T);
};

template <class T, int N, int EPT>
__global__ void __launch_bounds__(TlineCfg<T, N, EPT>::LAUNCH, TlineCfg<T, N, EPT>::SPLIT ? 2 : 1) tline_kernel(const TlineArgs A) {
    typedef TlineCfg<T, N, EPT> Cfg;
    typedef typename Cfg::S S;
    typedef cplx<T> C;
    constexpr int TPP = S::TPP, NT = Cfg::NT, TZ = Cfg::TZ;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* s_tw = reinterpret_cast<C*>(smem_raw);
    T* s_tab = reinterpret_cast<T*>(s_tw + N);                 // [full, half][N]
    C* s_x = reinterpret_cast<C*>(s_tab + 2 * N);              // exchange buffer of the transforms
    C* s_stash = s_x + (Cfg::SPLIT ? 2 : 1) * Cfg::XELEMS;     // [r][tid]: the half-branch input e4 q_s

    const int grp = threadIdx.x / NT, tid = threadIdx.x % NT;  // group 1 (SPLIT): the half branch of the step that starts
    for (int i = threadIdx.x; i < N; i += Cfg::LAUNCH) s_tw[i] = static_cast<const C*>(A.tw)[i];
    for (int i = threadIdx.x; i < 2 * N; i += Cfg::LAUNCH) s_tab[i] = static_cast<const T*>(A.tab[i / N])[i % N];
    const int ntile = A.plane / TZ, items = (ntile + Cfg::GPB_S - 1) / Cfg::GPB_S;
    const int b = A.b0 + blockIdx.x / items, idx = blockIdx.x % items, s = A.step;
    const int sp_now = species_index(A.packed, A.nspecies, A.seg, A.Ns, b, s), sp_prev = species_index(A.packed, A.nspecies, A.seg, A.Ns, b, s - 1);
    const bool cw = A.packed != 0, two = A.nprop == 2;
    // density pair of this slice (DensArgs)
    const int h = A.dens.half, jp = (two && b == 1) ? A.Ns - s : s;
    const bool dens = A.dens.on && (two ? (b == 0 ? s > h : s >= h) : s >= h), self = !two && s == h;
    double wA = 0.0, wB = 0.0, wA2 = 0.0, wB2 = 0.0;
    if (dens) {
        wA = A.dens.cA[jp]; wB = A.dens.cB[jp];
        if (cw) { if (!self) { wA2 = A.dens.cA[A.Ns - jp]; wB2 = A.dens.cB[A.Ns - jp]; } }
        else if (!two && !self) wA += A.dens.cA[A.Ns - jp];
    }
    __syncthreads();
    asm volatile("griddepcontrol.wait;" ::: "memory");         // everything below reads the previous kernel's output

    const int zz = tid % TZ, tb = tid / (TZ * TPP), t = (tid / TZ) % TPP;
    const int tile = idx * Cfg::GPB_S + tb;
    const bool active = tile < ntile;
    const long long base0 = (long long)tile * TZ + zz + (long long)t * A.plane, estride = (long long)A.plane * TPP;
    C* xs = s_x + grp * Cfg::XELEMS + tb * (N * TZ);
    const bool start = s < A.nsteps, keep = s <= A.dens.keep || s == A.nsteps;
    C* Fb = static_cast<C*>(A.F[b]); C* Hb = static_cast<C*>(A.H[b]);
    if (grp == 1) {                                            // H = Dx'[e4 q_s], as soon as group 0 has formed e4 q_s
        if (start) {
            asm volatile("bar.sync 3, %0;" ::"n"(2 * NT) : "memory");
            C v[EPT];
#pragma unroll
            for (int r = 0; r < EPT; ++r) v[r] = s_stash[r * NT + tid];
            diffuse<T, N, EPT, NT, typename Cfg::LS, typename Cfg::LC, 2>(v, t, zz, false, s_tw, s_tab + N, xs, xs);
            if (active) {
#pragma unroll
                for (int r = 0; r < EPT; ++r) stcg(Hb + base0 + r * estride, v[r]);
            }
        }
        asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
        return;
    }
    C* qs = static_cast<C*>(A.q[b]) + (long long)slice_slot(s, A.dens.keep) * A.M;
    const C* e4p = static_cast<const C*>(A.e4[sp_prev]); const C* e4n = static_cast<const C*>(A.e4[sp_now]);

    C v[EPT];
    if (s > 0) {                                               // finish step s-1:  q_s = (4 e4 Dx'[H] - F)/3   (Eq. 12)
#pragma unroll
        for (int r = 0; r < EPT; ++r) v[r] = active ? ldcg(Hb + base0 + r * estride) : mk<T>(0, 0);
        diffuse<T, N, EPT, NT, typename Cfg::LS, typename Cfg::LC>(v, t, zz, false, s_tw, s_tab + N, xs, s_x);
#pragma unroll
        for (int r = 0; r < EPT; ++r) {
            const C e = active ? ldcg(e4p + base0 + r * estride) : mk<T>(0, 0), f = active ? ldcg(Fb + base0 + r * estride) : mk<T>(0, 0);
            const C hh = cmul(v[r], e, cw);
            v[r] = mk<T>(((T)4 * hh.x - f.x) * (T)(1.0 / 3.0), ((T)4 * hh.y - f.y) * (T)(1.0 / 3.0));
        }
    } else {
#pragma unroll
        for (int r = 0; r < EPT; ++r) v[r] = mk<T>(1, cw ? 1 : 0);                   // q(x,0) = 1, q+(x,s=1) = 1; packed: 1 + i
    }
    if (keep && active) {
#pragma unroll
        for (int r = 0; r < EPT; ++r) stcg(qs + base0 + r * estride, v[r]);         // the slice store IS the step's output write
    }
    if (dens && active) {                                      // Eq. 8 (DensArgs): batched, all loads of a batch before its first store
        const C* partner = static_cast<const C*>(A.q[two ? 1 - b : 0]) + (long long)(A.Ns - s) * A.M;
        constexpr int BATCH = EPT < (sizeof(T) == 8 ? 4 : 8) ? EPT : (sizeof(T) == 8 ? 4 : 8);
        for (int pass = 0; pass < 2; ++pass) {
            const double w1 = pass == 0 ? wA : wB;
            if (cw ? pass == 1 : w1 == 0.0) continue;
            C* acc = static_cast<C*>(A.dens.acc[b][cw ? 0 : pass]);
#pragma unroll
            for (int r0 = 0; r0 < EPT; r0 += BATCH) {
                C zp[BATCH], a[BATCH];
#pragma unroll
                for (int k = 0; k < BATCH; ++k) {
                    const long long i = base0 + (r0 + k) * estride;
                    zp[k] = self ? v[r0 + k] : ldcg(partner + i);
                    a[k] = ldcg(acc + i);
                }
#pragma unroll
                for (int k = 0; k < BATCH; ++k) {
                    const long long i = base0 + (r0 + k) * estride;
                    const C q = v[r0 + k];
                    if (cw) {
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
    if (start) {                                               // start step s:  F = Dx[e2 q_s],  H = Dx'[e4 q_s]
#pragma unroll
        for (int r = 0; r < EPT; ++r) {
            const C e = active ? ldcg(e4n + base0 + r * estride) : mk<T>(0, 0);
            const C hb = cmul(v[r], e, cw);
            s_stash[r * NT + tid] = hb;
            v[r] = cmul(hb, e, cw);
        }
        if constexpr (Cfg::SPLIT) asm volatile("bar.arrive 3, %0;" ::"n"(2 * NT) : "memory");      // e4 q_s is in shared memory: group 1 takes the half branch
        diffuse<T, N, EPT, NT, typename Cfg::LS, typename Cfg::LC>(v, t, zz, false, s_tw, s_tab, xs, s_x);
        if (active) {
#pragma unroll
            for (int r = 0; r < EPT; ++r) stcg(Fb + base0 + r * estride, v[r]);
        }
        if constexpr (!Cfg::SPLIT) {
#pragma unroll
            for (int r = 0; r < EPT; ++r) v[r] = s_stash[r * NT + tid];
            diffuse<T, N, EPT, NT, typename Cfg::LS, typename Cfg::LC>(v, t, zz, false, s_tw, s_tab + N, xs, s_x);
            if (active) {
#pragma unroll
                for (int r = 0; r < EPT; ++r) stcg(Hb + base0 + r * estride, v[r]);
            }
        }
    }
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

}  // namespace fts
#endif
