// fts_plane.cuh — the y and z diffusions of one RQM4 step fused per yz-plane, for small grids (Ny = Nz = 16, 32 or 64).
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

}  // namespace fts
#endif
