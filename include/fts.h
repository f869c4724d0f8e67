/* fts.h — C ABI of fts-b200: the hot path of polymer field-theoretic simulation on one NVIDIA B200.
 *
 * Method: Delaney & Fredrickson, "Polymer Field-Theory Simulations on Graphics Processing Units",
 * arXiv 1204.5434 (text: PAPER.md, cited as PAPER.md:<line>).  The library solves the modified diffusion
 * equation (Eq. 5) for the chain propagators q and q+ with the 4th-order Richardson-extrapolated
 * pseudo-spectral step (Eq. 12), evaluates the single-chain partition function Q (PAPER.md:65
 * Eq. 4) and the segment volume fractions phi_A, phi_B (Eq. 8), and advances the fields by one
 * SCFT relaxation step or one complex-Langevin step (PAPER.md:102 Eq. 9, :112-118 Eq. 10-11).
 * Every step runs in hand-written sm_100a CUDA kernels; there is no CPU fallback and no cuFFT.
 *
 * Units and conventions: lengths in Rg, contour s in [0,1], ds = 1/Ns; the diffusion
 * factor is exp(-k^2 ds).  Grids: shape (Nx,Ny,Nz), layout [ix][iy][iz] with z contiguous, interleaved
 * (re,im); FTS_F64 = complex128, FTS_F32 = complex64.  Every grid dimension must be 1 or a power of two in
 * [8, 256] (FTS_EUNSUPPORTED otherwise; the paper benchmarks power-of-two grids); dimensions of 1
 * give the 1-D and 2-D problems of PAPER.md:193 (e.g. (N,1,1), (Nx,Ny,1)); 512 is not supported.
 *
 * Stored fields:  FTS_MODEL_EXTERNAL  f0 = w                       (one species in a given complex field)
 *                 FTS_MODEL_EDWARDS   f0 = Omega                   (chain feels i*Omega; Eq. 2)
 *                 FTS_MODEL_DIBLOCK   f0 = W+ = i*omega_+, f1 = W- = omega_-;  w_A = W+ - W-, w_B = W+ + W-
 *                                                                  (Eq. 3)
 *
 * Ownership: every *_dev pointer and the workspace are DEVICE memory allocated by the caller; the library
 * never allocates or frees device memory and keeps the workspace until fts_destroy.  Host outputs
 * (double[2] = re, im) are fp64 in both precisions.  `stream` is a cudaStream_t passed as void*.
 * All work is enqueued on `stream`; calls that return host scalars synchronise that stream.
 *
 * Errors: status codes only (no exceptions, no aborts); text of the last error from fts_last_error().
 * Determinism: same inputs and same (seed, step) give bit-identical outputs run to run (fixed-order
 * reductions, counter-based noise).
 */
#ifndef FTS_H
#define FTS_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct fts_ctx fts_ctx;

typedef enum {
    FTS_OK = 0,
    FTS_EINVAL = 1,        /* NULL pointer, Ns < 2, fA*Ns not an integer (1e-9), odd Simpson block, cell <= 0      */
    FTS_ESTATE = 2,        /* call order: fields not set, density before propagate, slice not retained           */
    FTS_EWORKSPACE = 3,    /* workspace smaller than fts_workspace_bytes, or not 256-byte aligned                   */
    FTS_ECUDA = 4,         /* a CUDA call failed; text in fts_last_error                                          */
    FTS_ENONFINITE = 5,    /* Q is NaN/Inf (diverged CL run)                                                       */
    FTS_EUNSUPPORTED = 6   /* grid dimension not 1 or a power of two in [8,256]; model/step combination not defined */
} fts_status;

typedef enum { FTS_F64 = 0, FTS_F32 = 1 } fts_precision;

typedef enum { FTS_MODEL_EXTERNAL = 0, FTS_MODEL_EDWARDS = 1, FTS_MODEL_DIBLOCK = 2 } fts_model;

typedef struct {
    int    model;                       /* fts_model                                                              */
    double fA, chiN, B, C;              /* block fraction, Flory parameter, excluded volume, chain density        */
    double lambda_plus, lambda_minus;   /* mobilities of Eq. 9 (Edwards uses lambda_plus); 0 is read as 1        */
    double noise_scale;                 /* multiplies eta in fts_cl_step: 1 = physical, 0 = deterministic         */
    int    store_both;                  /* 0: meet-in-the-middle store, slices 0..Ns/2 and the last one of q and of q+ are kept
                                           (half the memory); 1: every slice is kept (needed for Pi)          */
} fts_params;

/* Bytes of device workspace fts_create needs: fields, Boltzmann factors, the contour-slice store (Ns/2 + 2 slices per
 * propagator, or Ns + 1 with store_both; PAPER.md:183 memory analysis), density sums, scratch, tables. */
fts_status fts_workspace_bytes(const int grid[3], int Ns, const fts_params* params, fts_precision prec, size_t* bytes);

/* Builds the k-tables exp(-k_d^2 ds), exp(-k_d^2 ds/2) (once per simulation), the FFT
 * twiddles and the Simpson weights, and lays out the workspace.  cell = box lengths in Rg. */
fts_status fts_create(const int grid[3], const double cell[3], int Ns, const fts_params* params, fts_precision prec,
                      void* workspace_dev, size_t workspace_bytes, fts_ctx** out);
fts_status fts_destroy(fts_ctx* ctx);

/* Chain architecture of the two-species melt model (linear multiblock copolymers use the same
 * propagators): nblocks blocks listed from the s = 0 chain end, species[i] in {0 = A, 1 = B}, steps[i] contour steps
 * (even, >= 2, summing to Ns; host arrays).  Replaces the default AB diblock (fA Ns steps of A, then B): e.g. an ABA
 * triblock is species {0,1,0}.  q marches from s = 0, q+ from the far end; densities use Simpson's rule per block.
 * The SCFT / CL updates keep the homopolymer Debye kernel of Eq. 11 as their linear-response estimate.
 * FTS_EUNSUPPORTED for the one-species models.  Synchronises the device. */
fts_status fts_set_blocks(fts_ctx* ctx, int nblocks, const int* species, const int* steps);

/* Copy fields into / out of the context (device to device).  f1_dev is NULL for one-field models. */
fts_status fts_set_fields(fts_ctx* ctx, const void* f0_dev, const void* f1_dev, void* stream);
fts_status fts_get_fields(fts_ctx* ctx, void* f0_dev, void* f1_dev, void* stream);

/* PAPER.md:143 Boltzmann factors, then Ns RQM4 steps (Eq. 12) of q and, batched with it, q+ (diblock).  The march writes
 * the retained slices to the HBM store and accumulates the Simpson density sums of Eq. 8 as it goes: from the middle of
 * the chain on, each new slice is multiplied with the stored slice of the other propagator (meet-in-the-middle), so the
 * product is never written and no second pass over the store is needed.  Q = mean_x q(x,1) (Eq. 4) is left on the
 * device.  Asynchronous.  If the march gives up on an internal dependency (a bug or a lost SM; 5 s of wall clock) it stops,
 * Q becomes NaN and the next call that returns host scalars reports FTS_ECUDA; fts_set_fields clears that state. */
fts_status fts_propagate(fts_ctx* ctx, void* stream);
/* March only the first nsteps contour steps (truncated parity at 256^3); Q is then mean_x q_nsteps. */
fts_status fts_propagate_steps(fts_ctx* ctx, int nsteps, void* stream);

/* phi_A (and phi_B) = (ds/Q) sum_j c_j q_j q+_{Ns-j}, composite Simpson per block (Eq. 8; plain bilinear
 * product): normalises the sums the march accumulated.  Writes phi to caller memory, returns Q; synchronises
 * `stream`.  phiB_dev NULL for one species.  FTS_ESTATE before a full fts_propagate. */
fts_status fts_density_operators(fts_ctx* ctx, void* phiA_dev, void* phiB_dev, double Q_out[2], void* stream);

/* Copy slice j of q (which = 0) or q+ (which = 1; q+ is indexed from the far chain end) to out_dev.  Retained slices:
 * j <= Ns/2 and the last slice of the march (q(r,1) after a full march); all of them with store_both = 1.
 * FTS_ESTATE for a slice that was not retained or not reached. */
fts_status fts_get_slice(fts_ctx* ctx, int which, int j, void* out_dev, void* stream);

/* One SCFT iteration for the diblock melt (PAPER.md:84 forces; Eq. 11 at zero noise): W+ ascends with the
 * Debye-linearised response implicit, W- descends with its explicit linear term implicit.  seidel = 1
 * re-solves the propagators between the two updates (2 solves per iteration), seidel = 0 uses one solve.
 * H_out = H/(CV) of the fields at entry; resid_out = max|F+|, max|F-|.  Synchronises `stream`. */
fts_status fts_scft_step(fts_ctx* ctx, double dt_plus, double dt_minus, int seidel, double H_out[2], double resid_out[2], void* stream);

/* One complex-Langevin step (Eq. 9).  scheme 0 = Euler-Maruyama in real space; scheme 1 = the first-order
 * semi-implicit update of Eq. 10-11.  Noise: Philox4x32-10 keyed by `seed`, counter (site, step, field id),
 * Box-Muller, variance 2 lambda dt / dV, generated inside the update kernel.  Asynchronous. */
fts_status fts_cl_step(fts_ctx* ctx, double dt, int scheme, uint64_t seed, uint64_t step, void* stream);

/* Operators of the current fields; needs a completed fts_propagate - or a preceding fts_cl_step, in which case the
 * operators are those of the fields that step STARTED from, taken from the solve it already did (no further
 * propagator solve: operator averages over a CL run cost two small reductions per sample).  H: Eq. 2 (Edwards, extensive) or
 * Eq. 3 / (CV) (diblock); mu = ln C - ln Q; Pi: volume derivative of ln Z at fixed lattice fields (derived in
 * DESIGN.md, not printed in the paper: secondary output; needs store_both = 1, FTS_ESTATE otherwise).  Any pointer may be
 * NULL.  Synchronises `stream`. */
fts_status fts_operators(fts_ctx* ctx, double H[2], double mu[2], double Pi[2], void* stream);

/* Tuning options (integers), effective from the next fts_propagate / step call; the library reads NO environment
 * variables.  Unknown keys return FTS_EINVAL.  Keys:
 *   "march"       how the contour march is issued (fts_march_mode): 0 automatic (default), 1 one launch per phase and
 *                 step, 2 persistent ticket kernel with per-thread staging (fts_march.cuh), 3 persistent TMA kernel
 *                 (fts_march2.cuh; cubic grids of 128 or 256 points per side, FTS_EUNSUPPORTED otherwise)
 *   "slab_bytes"  mode 2: bytes of one L2 slab of the Y1/Z/Y2 phases (0 = one slab)
 *   "lag"         modes 2-3: slabs / planes between a phase and the phase that consumes it (-1 = default)
 *   "skew"        mode 3: planes by which q trails q+ inside a step (-1 = default)
 *   "interleave"  mode 2: alternate the two propagators' phases (default 1)
 *   "tz"          modes 1-2: pencils per strided tile, 8 or 16 (0 = default)
 *   "graph"       mode 1: replay the march's launches as one CUDA graph, captured once per context (default 1)
 *   "tline"       mode 1: straight-line kernel for the x pass of a step when Nx <= 64 (default 1)
 *   "plane"       mode 1: fuse the y and z passes of a step into one kernel per yz-plane when Ny = Nz = 16, 32 or 64 (default 1)
 *   "real_fields" 1: the caller declares that W+ and W- are real (SCFT; diblock only).  q and q+ are then
 *                 real and are marched together as ONE complex propagator z = q + i q+ (half the transforms and slices);
 *                 results agree with the general path to rounding; phi and slices are returned with zero imaginary part.
 *                 Fields that are not real make the next call that returns host scalars fail with FTS_EINVAL;
 *                 fts_cl_step (complex fields) is FTS_ESTATE and Pi FTS_EUNSUPPORTED while the option is set.
 * The march modes agree to rounding (the ticket kernel's variants are bit-identical among themselves). */
typedef enum { FTS_MARCH_AUTO = 0, FTS_MARCH_LAUNCH = 1, FTS_MARCH_TICKET = 2, FTS_MARCH_TMA = 3 } fts_march_mode;
fts_status fts_set_option(fts_ctx* ctx, const char* key, long long value);

/* Raw Philox4x32-10 block and the standard normal fts_cl_step draws for (seed, step, field, site), evaluated
 * ON THE DEVICE for n consecutive sites starting at site0; out_dev receives n doubles.  For tests. */
fts_status fts_debug_normals(uint64_t seed, uint64_t step, uint32_t field_id, uint64_t site0, size_t n, double* out_dev, void* stream);
/* The four raw 32-bit Philox4x32-10 words behind each of those normals (key = seed, counter = (site lo, site hi, step lo,
 * field_id ^ (step hi << 8)); reading A-15): out_dev receives 4 n words.  For the bit-exact test. */
fts_status fts_debug_philox(uint64_t seed, uint64_t step, uint32_t field_id, uint64_t site0, size_t n, uint32_t* out_dev, void* stream);

/* Measurement aids for bench.py.  fts_debug_fma_peak launches register-resident FMA chains (64 FMAs per thread per
 * iteration, 148*8 CTAs of 256 threads) and returns the number of FMAs issued, so the caller's own CUDA-event timing
 * gives the vector fp64/fp32 peak of this GPU; scratch_dev needs 148*8*256*8 bytes.  fts_launch_count returns the
 * number of kernels this library has launched since it was loaded. */
fts_status fts_debug_fma_peak(int precision, int iters, void* scratch_dev, size_t scratch_bytes, double* fma_count, void* stream);
uint64_t fts_launch_count(void);

/* Mean of a complex field without any caller-provided or library-allocated scratch: mean_dev[0..1] = (re, im) of
 * (1/npoints) sum_x field[x], accumulated in fp64.  With field = the last contour slice q(x,1) this is Q of PAPER.md:65
 * Eq. 4, computed with the same fixed-order two-stage sum as fts_propagate (bit-identical to the Q it leaves behind).
 *
 * Why it exists: everything else in this header works inside the workspace handed to fts_create.  A caller may have no
 * such memory to give and no way to get any - an observer inside another program's run that receives slice pointers
 * but owns no context while the host program has already split all of HBM among its own buffers; code on a path where
 * marches are in flight on other streams and the device-wide synchronisation cudaMalloc / cudaFree can cause is not
 * acceptable; a process whose allocator must not see raw runtime allocations next to its pool.  For those the per-CTA
 * partial sums live in a fixed array inside the library's device image (9472 bytes on every GPU that loads libfts.so,
 * held until the process exits).  This call never calls cudaMalloc, cudaFree or any allocating routine.
 *
 * Arguments: field_dev - DEVICE, npoints interleaved (re, im) pairs of the given precision, read only; mean_dev - DEVICE,
 * two doubles, written on `stream`; both stay the caller's.  errbuf (HOST, may be NULL) receives a NUL-terminated
 * message of at most errbuf_len bytes when the status is not FTS_OK.  Asynchronous: nothing is synchronised.
 * Limit: npoints <= FTS_MEAN_NOALLOC_MAX_POINTS (256^3, the largest grid of this library); above it FTS_EUNSUPPORTED with
 * a message, nothing launched.  FTS_EINVAL: NULL field_dev / mean_dev, npoints = 0, unknown precision.  FTS_ECUDA: the
 * address look-up or a launch failed.
 * First call per device: looks up the array's device address once, with the current device (this can initialise the
 * CUDA context and load the device code) - make it at start-up, with the intended device current, before any stream
 * capture on that device.  Later calls only enqueue two small kernels on the current device.
 * Shared state: every call on a device uses the same array.  Nothing in it needs zeroing (each call overwrites exactly
 * the partials it then reads), but calls that can overlap on one GPU - different streams, or host threads using
 * different streams - race on it and return wrong means.  Keep them on one stream or order them with events.
 * Not counted by fts_launch_count. */
#define FTS_MEAN_NOALLOC_MAX_POINTS 16777216
fts_status fts_mean_noalloc(const void* field_dev, size_t npoints, fts_precision prec, double* mean_dev, void* stream,
                            char* errbuf, size_t errbuf_len);

const char* fts_last_error(const fts_ctx* ctx);
const char* fts_version(void);

#ifdef __cplusplus
}
#endif
#endif
