/* fts_oracle.h — C ABI of the CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, single-threaded CPU implementation of the discretised scheme of
 * Delaney & Fredrickson, "Polymer Field-Theory Simulations on Graphics Processing Units"
 * (arXiv 1204.5434; text in /root/reference/PAPER.md, cited below as PAPER.md:<line>).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load this library.  It shares no code with the CUDA library (paper_1204_5434_b200/csrc):
 * own FFT, own Philox, own tables, own Simpson weights.  All pointers are HOST pointers.
 *
 * Conventions: lengths in Rg, contour s in [0,1], ds = 1/Ns,
 * grid layout [ix][iy][iz] with z contiguous, interleaved (re,im); precision 0 = complex128,
 * 1 = complex64 (all arithmetic in float, tables computed in double then rounded).
 * Stored fields: model 0 (external)  f0 = w;
 *                model 1 (Edwards)   f0 = Omega            (chain feels i*Omega, Eq. 2);
 *                model 2 (diblock)   f0 = W+ = i*omega_+,  f1 = W- = omega_-   (Eq. 3).
 *
 * Pins (tests/test_oracle_pins.py): direct DFT, uniform-field closed form, dense 4^3 operator and
 * dense matrix exponential, 4th-order convergence, mean_x q_j q+_{Ns-j} = Q, Debye response,
 * homogeneous saddles (diblock H, Edwards H/mu/Pi), Philox known-answer vectors; the SCFT multipliers and the
 * Eq. 10-11 (scheme 1) update, both models, to the backward-Euler / IMEX step of the linearised dynamics and to
 * exactly filtered noise at the saddle.  The Pi operator (derived, reading A-14: the paper prints no formula) is pinned by
 * its mean-field values and by finite-difference d ln Q/dV of its K term on both branches: one species, and the diblock
 * with complex fields and unequal blocks (q+ != q), where the pin also rejects q_{Ns-j} or q+_j in place of q+_{Ns-j}.
 */
#ifndef FTS_ORACLE_H
#define FTS_ORACLE_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct oracle_ctx oracle_ctx;

typedef struct {
    int    model;            /* 0 external, 1 Edwards, 2 diblock                                   */
    double fA, chiN, B, C;   /* unused ones ignored                                                */
    double lambda_plus, lambda_minus;   /* mobilities (Edwards uses lambda_plus)                   */
    double noise_scale;      /* multiplies eta; 1 = physical CL noise, 0 = deterministic relaxation */
    int    store_both;       /* ignored by the oracle: it always keeps every slice                 */
} oracle_params;

/* returns 0 on success, nonzero = same numbering as fts_status (1 EINVAL, 2 ESTATE, 6 EUNSUPPORTED) */
int  oracle_create(const int grid[3], const double cell[3], int Ns, const oracle_params*, int precision, oracle_ctx** out);
void oracle_destroy(oracle_ctx*);
int  oracle_set_fields(oracle_ctx*, const void* f0, const void* f1);
int  oracle_get_fields(oracle_ctx*, void* f0, void* f1);
/* O2-O7: Boltzmann factors, forward and conjugate march (Eq. 12 per step), Q (Eq. 4). */
int  oracle_propagate(oracle_ctx*);
/* march only the first nsteps contour steps (truncated parity at 256^3); Q is then mean(q_nsteps). */
int  oracle_propagate_steps(oracle_ctx*, int nsteps);
/* O8: phi_A, phi_B (Eq. 8, composite Simpson per block), Q. phiB may be NULL for one species. */
/* Linear AB multiblock chain: blocks from the s = 0 end, species[i] in {0 = A, 1 = B}, steps[i] even, sum = Ns.
 * Diblock model only (6 otherwise); replaces the default (fA Ns of A, then B).  Densities use Simpson's rule per block. */
int  oracle_set_blocks(oracle_ctx*, int nblocks, const int* species, const int* steps);
int  oracle_density_operators(oracle_ctx*, void* phiA, void* phiB, double Q_out[2]);
int  oracle_get_slice(oracle_ctx*, int which, int j, void* out);
int  oracle_scft_step(oracle_ctx*, double dt_plus, double dt_minus, int seidel, double H_out[2], double resid_out[2]);
int  oracle_cl_step(oracle_ctx*, double dt, int scheme, uint64_t seed, uint64_t step);
int  oracle_operators(oracle_ctx*, double H[2], double mu[2], double Pi[2]);

/* ---- exposed building blocks, so that each can be pinned on its own ---- */
/* unnormalised forward (sign=-1) / inverse-with-1/n (sign=+1) 1-D DFT, radix-2 when n is a power of two */
void oracle_fft1d(double* data_interleaved, int n, int sign);
/* the same transform by the O(n^2) definition */
void oracle_dft1d_direct(double* data_interleaved, int n, int sign);
/* one Eq. 12 step applied to an arbitrary q with an arbitrary species field w (complex128, M entries each) */
int  oracle_rqm4_step(const int grid[3], const double cell[3], double ds, const void* w, const void* q_in, void* q_out);
/* Philox4x32-10 (Salmon et al., SC'11): counter c[4], key k[2] -> out[4] */
void oracle_philox4x32_10(const uint32_t c[4], const uint32_t k[2], uint32_t out[4]);
/* the standard normal the CL step draws for (seed, step, field id, site)  (reading A-15) */
double oracle_normal(uint64_t seed, uint64_t step, uint32_t field_id, uint64_t site);
/* Debye function g_D(x) = 2(exp(-x)+x-1)/x^2, g_D(0)=1 */
double oracle_debye(double x);

#ifdef __cplusplus
}
#endif
#endif
