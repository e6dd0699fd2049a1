/*
 * tkhp.h -- C ABI of libtkhp: real-space AMOEBA polarization on one NVIDIA B200.
 *
 * Hot path of arXiv 2011.01207 (Tinker-HP on GPUs; "P:Lnnn" = PAPER.md line nnn):
 *   blocked neighbour list  ->  permanent-multipole field  ->  induced-dipole
 *   T.mu matrix-vector product inside a Jacobi-preconditioned CG solve  ->
 *   polarization energy.
 * The paper gives the organisation (32-atom groups and a group-pair list, P:L296-366;
 * list filtering to a group->atom list with phantom atoms; pair kernels
 * that compute every pair unscaled and apply the few scaling factors in a separate
 * pass; PCG with a diagonal preconditioner, one polarization matrix-vector
 * product per iteration; FP32 pair math with FP64 accumulation,
 * P:L263-279).  It prints no interaction formula; the arithmetic is the standard
 * AMOEBA real-space Ewald field with exponential Thole damping, written out in
 * DESIGN.md section 2 (equations F1-F3, T1-T2, S, U), which restates SURVEY.md 8(c).
 *
 * Conventions (all entry points)
 *   - Units: Angstrom, elementary charge, Angstrom^3; energy in kcal/mol.
 *   - Every user-facing array is FP64, in ORIGINAL atom order (the spatial sort is
 *     internal), C-contiguous.  Pointers named d_* are CUDA DEVICE pointers owned by
 *     the caller; pointers named h_* are HOST pointers owned by the caller.
 *   - `stream` is a cudaStream_t passed as void* (0 = legacy default stream).  Calls
 *     are asynchronous on `stream` unless the comment says "synchronises".
 *   - Return value: TKHP_OK (0) or a negative TKHP_E* code; nothing is thrown across
 *     the ABI.  After an error the contents of output arrays are unspecified and
 *     tkhp_last_error() describes the failure.
 *   - No allocation after tkhp_create(): all device memory is the caller's workspace.
 *   - A context is not thread-safe; use one per host thread / stream.
 *   - There is no CPU fallback: without a CUDA device tkhp_create() fails (TKHP_ECUDA).
 */
#ifndef TKHP_H
#define TKHP_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tkhp_ctx tkhp_ctx; /* opaque; owned by the library */

enum {
    TKHP_OK = 0,
    TKHP_EINVAL = -1,     /* bad argument / parameter out of the supported range */
    TKHP_ECUDA = -2,      /* CUDA runtime error or no device */
    TKHP_ECUTOFF = -3,    /* cutoff + skin > box/2 (single minimum image only) */
    TKHP_ENOLIST = -4,    /* tkhp_nblist_build() has not been called on this context */
    TKHP_ENOCONV = -5,    /* PCG hit max_iter; d_mu holds the best iterate */
    TKHP_ECAPACITY = -6,  /* workspace too small for this geometry (see max_* params) */
    TKHP_ENONFINITE = -7  /* NaN/Inf in positions, or polarizability <= 0 */
};

/* precision of the pair arithmetic (DP and MP modes) */
enum {
    TKHP_FP64 = 0,  /* every operation in FP64 */
    TKHP_MIXED = 1, /* FP32 pair math, FP64 accumulation of fields and of all dot products */
    TKHP_FIXED = 2  /* the paper's FP mode (eqs 2-3): FP32 pair math as in MIXED, the
                       64-bit containers of the pair kernels are INTEGERS, a = int(round(x 2^fB)) with
                       fB = 34 fractional bits for the field and T.mu accumulators and 30 for the
                       energy (round = to nearest); PCG dot products stay FP64 tree reductions */
};

/* which pair-list the compute kernels walk (both are built from the same 32-atom blocks) */
enum {
    TKHP_LIST_TILES = 0,   /* one warp per 32x32 block pair of the block-pair list */
    TKHP_LIST_CLUSTER = 1, /* filtered 8-atom-cluster -> atom lists, the paper's "list filtering"
                               at finer granularity; falls back to TILES when the
                              box is too small for it (box/2 < cutoff + block extent) */
    TKHP_LIST_ATOM = 2     /* the filtering carried to the end: one exact list per atom (every entry
                              is a pair inside r_c for the positions of the build), stored
                              lane-interleaved per 32-atom block; built from the CLUSTER lists.
                              Falls back to CLUSTER (then TILES) when a capacity is exceeded */
};

typedef struct {
    int32_t n_atoms;     /* N >= 1 */
    int32_t precision;   /* TKHP_FP64 | TKHP_MIXED | TKHP_FIXED */
    int32_t device;      /* CUDA device ordinal */
    int32_t list_mode;   /* TKHP_LIST_TILES | TKHP_LIST_CLUSTER | TKHP_LIST_ATOM */
    double box;          /* cubic box edge L; <= 0: open boundary, no images (tests) */
    double cutoff;       /* r_c: a pair contributes iff R^2 <= r_c^2 */
    double skin;         /* list buffer: block pairs kept by box distance <= r_c + skin */
    double ewald_beta;   /* Ewald coefficient beta (1/A); 0: bare Coulomb, no self term (tests) */
    double thole_a;      /* Thole width a (0.39 for AMOEBA water) */
    int32_t max_tiles_per_block; /* capacity of the block-pair list per block; 0 = automatic */
    int32_t max_nbrs_per_cluster; /* capacity of a cluster's atom list; 0 = automatic */
    int32_t max_nbrs_per_atom;   /* ATOM mode: capacity of one atom's list incl. padding; 0 = automatic */
    int32_t max_stage_per_chunk; /* ATOM mode: staged atoms per shared-memory chunk (multiple of 32);
                                    0 = automatic (what fits the kernel's shared memory); tests use a
                                    small value to exercise the multi-chunk path */
    int32_t solver_flags;        /* OR of TKHP_SOLVER_*; 0 = automatic (tests use the flags to force the
                                    fall-back paths of tkhp_polar_solve) */
    int32_t reserved;            /* must be 0 */
} tkhp_params;

/* tkhp_params.solver_flags */
enum {
    TKHP_SOLVER_NO_PERSISTENT = 1, /* never run the solve as one persistent cooperative kernel (k_pcg_persist: MIXED/
                                      FIXED precision, ATOM lists, every group's neighbourhood in one chunk, grid
                                      co-resident; k_pcg_tiles: TILES mode, at most 16,384 padded atoms, any
                                      precision); the launch-per-matvec loop is used instead */
    TKHP_SOLVER_NO_FUSED_STEP = 2, /* launch-per-matvec path: update and direction as two kernels */
    TKHP_SOLVER_STORED_T = 4,      /* MIXED/FIXED precision, ATOM lists: precompute the real-space matrix elements
                                      (two radial factors per list slot, 8 bytes) after a list build and stream
                                      them in every T.mu product instead of re-evaluating the
                                      radial functions; tkhp_tmatvec and the launch-per-matvec solve use it, the
                                      persistent solve kernel is not used.  Adds 8 bytes per list slot of capacity
                                      to the workspace. */
    TKHP_SOLVER_TEST_BARRIER_FAULT = 8 /* tests only: the last CTA of a persistent solve kernel returns before its first
                                      grid barrier, as a CTA lost to a fault would.  The others give up after 2 s, the
                                      kernel leaves d_mu untouched, and tkhp_polar_solve repeats the solve on the
                                      launch-per-matvec path (as after any barrier time-out) and keeps to that path */
};

/* Bytes of device workspace tkhp_create() needs for these parameters.  Host, pure. */
int tkhp_workspace_bytes(const tkhp_params *params, size_t *bytes);

/* Create a context on params->device using caller-owned device memory d_workspace
 * (>= tkhp_workspace_bytes, 256-byte aligned).  Synchronises.  *out is NULL on error. */
int tkhp_create(const tkhp_params *params, void *d_workspace, size_t bytes, tkhp_ctx **out);
int tkhp_destroy(tkhp_ctx *ctx);

/* Text of the last error on this context (ctx-owned, valid until the next call);
 * with ctx == NULL: the last error of a failed tkhp_create() (or of a context-free call such as
 * tkhp_polar_energy_static) on this thread. */
const char *tkhp_last_error(const tkhp_ctx *ctx);

/*
 * Neighbour list (P:L310-366 cells -> groups of B_size = 32 -> group-pair list;
 * BASELINE.json north_star: "atoms are sorted spatially into 32-atom blocks, and block
 * pairs are kept by bounding-box distance against the cutoff plus a skin").
 *   d_pos            N*3  positions (x,y,z per atom), any image
 *   d_polarizability N    alpha_i > 0
 *   d_group_id       N    polarization group, 0 <= g < N (same group => masked pair)
 * Steps: wrap, Hilbert cell key on a 2^b grid, stable sort by (key, index), gather to
 * block-local structure-of-arrays, per-block bounding boxes, block pairs (I <= J) with
 * box gap^2 <= (cutoff+skin)^2 (FP64, no FMA contraction: DESIGN.md section 3), and, in
 * CLUSTER and ATOM mode, the filtered cluster->atom lists and the exact per-atom lists
 * at r_c.  The positions passed here are the positions every later call on this context
 * uses.
 * Coincident atoms: the finer lists identify an atom with itself by R^2 <= 1e-10 A^2, so
 * two DISTINCT atoms closer than 1e-5 A do not interact in CLUSTER/ATOM mode (they would
 * give 1/0 in the pair formulas; the TILES kernels and the oracle skip only i == j).
 * Polarization groups are expected to be small (molecules): the mask-correction pass
 * walks all mates of an atom's group on one thread.
 * On a stream of the caller's (not the legacy default stream 0) the whole build is
 * captured once into a CUDA graph, keyed by the three input pointers, and replayed by
 * later calls with the same pointers; contents may change freely between calls.  The graphs
 * of the four most recently used pointer triples are kept (an integrator that alternates
 * between position buffers does not re-capture); a fifth triple replaces the least recently
 * used one.  If `stream` is being captured by the caller, or a capture ever fails, the build
 * is enqueued as plain launches instead; tkhp_profile_read_build() counts each case.
 */
int tkhp_nblist_build(tkhp_ctx *ctx, const double *d_pos, const double *d_polarizability,
                      const int32_t *d_group_id, void *stream);

/* Read-only view of the list.  Synchronises `stream`.  Pointers stay valid until the
 * next tkhp_nblist_build()/tkhp_destroy().
 *   *d_perm   32*n_blocks int32: original atom index per sorted slot, -1 = phantom
 *             (phantoms only at the end of the last block)
 *   *d_pairs  2*n_pairs int32: (I,J), I <= J, sorted lexicographically            */
int tkhp_nblist_view(tkhp_ctx *ctx, int32_t *n_blocks, int64_t *n_pairs,
                     const int32_t **d_perm, const int32_t **d_pairs, void *stream);

/* Statistics of the current list.  Synchronises `stream`.  Any pointer may be NULL.
 *   n_pairs_within_cutoff  unordered atom pairs {i,j}, i != j, R^2 <= r_c^2 (FP64 test):
 *                          the "useful pair interactions" of one field / T.mu evaluation
 *   n_slots_evaluated      lane-slots the compute kernels of the active list mode walk
 *                          per evaluation (tiles: 1024 per off-diagonal tile, 992 per
 *                          diagonal tile; cluster: 8 x list length summed over clusters;
 *                          atom: 32 x padded list length summed over blocks)
 *   list_mode_in_use       TKHP_LIST_TILES, _CLUSTER or _ATOM after any fallback     */
int tkhp_nblist_stats(tkhp_ctx *ctx, int64_t *n_pairs_within_cutoff, int64_t *n_slots_evaluated,
                      int32_t *list_mode_in_use, void *stream);

/* Break-down of the ATOM lists ("list filtering", carried down to the atom; DESIGN.md
 * section 5.3).  Synchronises `stream`.  out[0] = lane-slots in FAR rows (pairs evaluated without
 * the Thole term), out[1] = lane-slots in NEAR rows (full formula), out[2] = list segments summed
 * over blocks, out[3] = 1 if the far class is in use (MIXED precision and ewald_beta > 0), else 0
 * (then every slot is counted in out[0] and evaluated with the full formula).  All zero unless
 * the list mode in use is TKHP_LIST_ATOM.  TKHP_ENOLIST before a build.                      */
int tkhp_nblist_atom_stats(tkhp_ctx *ctx, int64_t out[4], void *stream);

/*
 * Permanent-multipole field (F1-F3; charge, dipole, traceless quadrupole,
 * erfc-damped real-space Ewald with Thole damping; same-group pairs masked; Ewald self
 * term on d_i).  "Same strategy for the other real space kernels (electrostatics and
 * polarization)"; masked pairs in a separate FP64 pass.
 *   d_charge N, d_dipole N*3, d_quad N*6 (xx,xy,xz,yy,yz,zz; traceless Cartesian),
 *   d_field  N*3 out (e/A^2).
 */
int tkhp_perm_field(tkhp_ctx *ctx, const double *d_charge, const double *d_dipole,
                    const double *d_quad, double *d_field, void *stream);

/* d_out = T_real d_mu + (4 beta^3 / (3 sqrt(pi))) d_mu   (T1-T2; "the matrix-vector
 * product").  d_mu, d_out: N*3; must not alias. */
int tkhp_tmatvec(tkhp_ctx *ctx, const double *d_mu, double *d_out, void *stream);

/*
 * Solve (alpha^-1 - T) mu = field by conjugate gradients with the diagonal (Jacobi)
 * preconditioner alpha (recurrences in DESIGN.md S).
 *   d_field   N*3 right-hand side
 *   d_mu      N*3 in: initial guess if use_guess != 0 (else alpha*field is used); out: mu
 *   tol       stop when sqrt(sum_i |r_i|^2 / N) < tol  (e/A^2)
 *   h_iters   host out: number of T.p products in the loop;  h_rms host out: final rms
 * Synchronises `stream` (convergence is read back by the host).  Returns TKHP_ENOCONV
 * (with the best mu) when max_iter is reached.
 * The persistent solve kernels synchronise their CTAs with grid barriers that give up after 2 s
 * (%globaltimer).  A solve whose barrier broke writes nothing to d_mu; the call then repeats it
 * with one launch per product, and the context uses that path from then on
 * (tkhp_profile_read_build out[4] counts these events).
 */
int tkhp_polar_solve(tkhp_ctx *ctx, const double *d_field, double *d_mu, double tol,
                     int32_t max_iter, int32_t use_guess, int32_t *h_iters, double *h_rms,
                     void *stream);

/* *d_energy (device, 1 double) = -1/2 * 332.063713 * sum_i mu_i . field_i  (kcal/mol). */
int tkhp_polar_energy(tkhp_ctx *ctx, const double *d_mu, const double *d_field,
                      double *d_energy, void *stream);

/*
 * The same energy for callers that cannot allocate: no context, no workspace, no cudaMalloc.
 *
 * Who this is for.  Every other call needs a tkhp_ctx, and tkhp_create() needs a workspace that
 * somebody obtained from cudaMalloc (it also creates streams, events and pinned host buffers).
 * Code that runs where allocation is off limits cannot provide that: a force-field plug-in called
 * from inside an MD engine's step loop after the engine has given all device memory to its own
 * pool; a callback that runs while another host thread has a stream capture open, when the CUDA
 * runtime refuses cudaMalloc; a step loop that cannot afford the device-wide stall of
 * cudaMalloc/cudaFree.  Such a caller already holds mu and the field on the device and wants
 * E_pol = -1/2 * 332.063713 * sum_i mu_i . field_i in *d_energy (device, 1 double, kcal/mol).
 *
 *   device    CUDA device ordinal that owns d_mu, d_field, d_energy and `stream` (0..63)
 *   n_atoms   1 <= n_atoms <= TKHP_STATIC_MAX_ATOMS; d_mu, d_field: n_atoms*3 FP64, any atom order
 *
 * The block partial sums and the ticket counter of the reduction live in an 8,448-byte array that is
 * part of the library's device image (a file-scope __device__ array in csrc/energy_static.cu): every
 * GPU that loads libtkhp holds these bytes until the process exits, and this call neither creates nor
 * frees anything -- it calls no cudaMalloc, cudaFree, cudaHostAlloc or allocating library routine.
 * The scratch is sized for 1,024 partial sums; beyond TKHP_STATIC_MAX_ATOMS (2^22, four times the
 * paper's largest system) the call is refused with TKHP_ECAPACITY and leaves *d_energy untouched.
 *
 * First call on a device: looks up the array's device address (cudaGetSymbolAddress, which also makes
 * the CUDA runtime load the library's device code on that GPU).  That is host-side set-up, done once
 * per device under a mutex; make this first call before you begin any stream capture.
 *
 * Sharing: all calls on a GPU use the same array, which keeps whatever the previous call left.  The
 * call clears the ticket on `stream` before the kernel; the partials need no clearing.  Two calls
 * that can overlap on the GPU (different streams without an ordering between them, or different host
 * threads on the same device) race on the array and give wrong energies: order them.
 *
 * Asynchronous on `stream`; leaves the caller's current device as it found it.  The value is that of
 * tkhp_polar_energy on an FP64 or MIXED context, same summation order (TKHP_FIXED contexts round every
 * term to 2^-30 kcal/mol first; this call does not).  Errors: TKHP_EINVAL (NULL pointer, n_atoms < 1,
 * device ordinal), TKHP_ECAPACITY (n_atoms too large), TKHP_ECUDA; tkhp_last_error(NULL) has the text.
 */
#define TKHP_STATIC_MAX_ATOMS 4194304
int tkhp_polar_energy_static(int32_t device, int64_t n_atoms, const double *d_mu, const double *d_field,
                             double *d_energy, void *stream);

/*
 * Whole hot path from HOST buffers (end-to-end entry used for the e2e benchmark leg):
 * copies the inputs to the device, builds the list, evaluates the field, solves for mu,
 * computes E_pol and copies mu, field and E_pol back.  Host arrays as in the calls above.
 * The staging buffers come from the context's workspace; the multipole copies run on a stream of
 * the context beside the list build.  Synchronises.
 */
int tkhp_polarize_host(tkhp_ctx *ctx, const double *h_pos, const double *h_polarizability,
                       const int32_t *h_group_id, const double *h_charge, const double *h_dipole,
                       const double *h_quad, double tol, int32_t max_iter,
                       double *h_mu /* N*3 out, may be NULL */,
                       double *h_field /* N*3 out, may be NULL */, double *h_energy /* 1 out */,
                       int32_t *h_iters, double *h_rms, void *stream);

/* Timing of the internal phases of the most recent call that ran them, in ms, measured with
 * CUDA events on the call's stream: [0] list build, [1] field, [2] last T.mu kernel,
 * [3] solve, [4] energy.  Synchronises the events.  Any entry not run yet is < 0. */
int tkhp_last_timings(tkhp_ctx *ctx, double ms[5]);

/*
 * Launch accounting and live kernel timing for benchmarks.
 * tkhp_profile_reset zeroes the launch counter; with enable_kernel_events != 0 every later
 * T.mu / field PAIR kernel launch (at most 64 of each until the next reset) is bracketed by
 * its own CUDA event pair on the launching stream.  tkhp_profile_read synchronises those
 * events and returns: kernels launched by this context since the reset (every __global__
 * launch of libtkhp; memsets and copies are not kernels), the number of recorded T.mu pair
 * kernel launches and their summed duration in ms, the same for the field pair kernel.
 * Any output pointer may be NULL.
 */
int tkhp_profile_reset(tkhp_ctx *ctx, int32_t enable_kernel_events);
int tkhp_profile_read(tkhp_ctx *ctx, int64_t *n_kernel_launches, int32_t *n_tmatvec_kernels,
                      double *tmatvec_kernel_ms, int32_t *n_field_kernels, double *field_kernel_ms);
/* The same for the persistent PCG kernels (k_pcg_persist, k_pcg_tiles: the whole solve is one
 * cooperative launch): recorded launches since the reset, their summed
 * duration in ms and the T.mu products they performed (iterations + 1 per solve). */
int tkhp_profile_read_solve(tkhp_ctx *ctx, int32_t *n_solve_kernels, double *solve_kernel_ms, int64_t *n_matvecs);
/* How the list builds of this context ran since tkhp_create (host counters, no synchronisation):
 * out[0] = build graphs captured and instantiated (each costs far more host time than a replay saves:
 * a number that grows with every build means the caller passes ever new pointers), out[1] = builds
 * replayed from a cached graph, out[2] = builds enqueued as plain launches (legacy stream 0, caller's
 * stream under capture, or graphs switched off), out[3] = 1 if a failed capture has switched graphs
 * off for this context; and, kept with them although it concerns the solve, out[4] = persistent solves
 * abandoned on a broken grid barrier and repeated on the launch-per-matvec path. */
int tkhp_profile_read_build(tkhp_ctx *ctx, int64_t out[5]);

/*
 * Register-resident FMA microbenchmark used as the measured ALU roofline denominator
 * (SURVEY 8(d) "Peaks"): runs dependent-chain FMAs with 8 accumulators per thread on every
 * SM for about `seconds`, returns sustained TFLOP/s (2 flops per FMA).
 *   precision: TKHP_MIXED -> FP32 FFMA, TKHP_FP64 -> DFMA.   Synchronises.
 * A benchmark helper outside the "no allocation after tkhp_create()" rule: it needs no context,
 * makes `device` current for the measurement (the caller's current device is restored on return)
 * and allocates and frees one scalar with cudaMalloc/cudaFree and two events.
 */
int tkhp_fma_peak(int32_t device, int32_t precision, double seconds, double *tflops);

#ifdef __cplusplus
}
#endif
#endif /* TKHP_H */
