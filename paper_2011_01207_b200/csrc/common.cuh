// common.cuh -- context, workspace layout and small helpers shared by the .cu files of libtkhp.
// B200 / sm_100a only.  No code here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "../../include/tkhp.h"

namespace tkhp {

constexpr int BLOCK = 32;          // B_size: atoms per block = warp size
constexpr int CLUSTER = 8;         // atoms per cluster in CLUSTER list mode
constexpr int SUPER = 32;          // blocks per super-block in the hierarchical pair search
constexpr int MAX_PARTIALS = 1024; // reduction partials per dot product
constexpr double COULOMB = 332.063713;          // kcal A / (mol e^2)  (DESIGN.md U)
constexpr double SQRT_PI = 1.772453850905516027298167483341;
constexpr float PHANTOM_FAR = 1.0e6f;            // local coordinate of phantom atoms (A)

// Device-resident scalars written by kernels and read by later kernels or by the host.
struct DeviceState {
    // error flags (sticky until the next build)
    int err_nonfinite;      // NaN/Inf position
    int err_bad_alpha;      // alpha <= 0
    int err_bad_group;      // group id outside [0, N)
    int err_capacity;       // tile list or cluster list overflow
    int err_barrier;        // a grid barrier of a persistent PCG kernel timed out (diagnostic, sticky until the next build;
                            // the kernels report a broken barrier through their result slot, not through this flag)
    int pad_err;
    // grid (sort key)
    int grid_bits;          // b
    int pad0;
    double grid_origin[3];  // 0 when periodic, per-axis minimum when open
    double grid_inv_h;      // 2^b / extent
    double lo[3], hi[3];    // open-boundary extent reduction
    // geometry
    unsigned long long max_half_bits;   // max block half-extent over all axes (bits of a double >= 0)
    int per_pair_image;                 // 1: box too small for one image shift per tile
    int cluster_bad;                    // 1: CLUSTER lists unusable (box too small / capacity): TILES are used
    int max_stage;                      // largest staged-atom count of any group (CLUSTER mode)
    // list sizes
    long long n_tiles;                  // block pairs kept
    long long n_diag_tiles;
    long long n_cluster_entries;        // total entries of all cluster lists (CLUSTER mode)
    long long n_pairs_within_cutoff;    // statistics (tkhp_nblist_stats)
    long long n_atom_entries;           // ATOM mode: padded per-lane list entries summed over blocks
    long long n_atom_far;               //   of which in FAR rows
    long long n_atom_segments;          // ATOM mode: list segments summed over blocks
    int atom_bad;                       // 1: ATOM lists unusable (capacity / too many chunks): CLUSTER is used
    int pad1;
    // PCG scalars
    double rzv[2];          // r.z ping-pong (iteration parity)
    double pq, rr, gamma, delta;
    unsigned ticket;        // last-block reductions (reduce.cuh); 0 between kernels
    int bar_gen;            // grid barrier of k_pcg_step: the iteration whose partial sums are complete
    unsigned long long energy_fixed;   // TKHP_FIXED: int64 container of the energy (30 fractional bits), 0 between kernels
    unsigned bar_count;     // grid barrier of k_pcg_persist: arrivals (monotonic within a solve) ...
    unsigned bar_release;   // ... and the last barrier every CTA has reached (adjacent: zeroed together)
    int conv_at;            // PCG: iterations with index >= conv_at are skipped on the device
    int iters;
};

struct Ctx {
    tkhp_params p;
    int n, n_blocks, n_pad, n_super;
    int sm_count;
    bool built;
    int list_mode_in_use;
    long long cap_tiles;
    long long n_tiles_host;             // valid after a view/stats/solve sync
    int n_cells_alloc;                  // 2^(3 b_alloc)
    int grid_bits_host;                 // periodic: b ; open: -1 (computed on device)
    char err[512];

    // ---- workspace carve (device pointers) ----
    DeviceState *st;
    // sort
    uint32_t *key;          // N
    uint32_t *cell_count;   // n_cells_alloc + 1  (also reused for group histogram: needs >= N+1)
    uint32_t *cell_start;   // n_cells_alloc + 1
    uint32_t *scan_tmp;     // block sums for the scan
    int32_t *tmp_idx;       // N
    // scratch of the polarization-group sort, which runs beside the spatial sort (side stream / graph branch)
    uint32_t *key2, *count2, *scan_tmp2;   // N, N + 2, block sums
    int32_t *tmp_idx2;      // N
    int32_t *perm;          // n_pad, -1 = phantom
    // copies of the caller's build inputs in ORIGINAL order (the list is valid for these positions)
    double *pos_o;          // 3 N
    int32_t *group_o;       // N
    // polarization groups (mask correction)
    uint32_t *grp_start;    // N + 1
    int32_t *grp_members;   // N
    // sorted, block-local structure of arrays
    float4 *xyzw32;         // n_pad: local x,y,z (A), w = (a/alpha)^(1/2)
    double4 *xyzw64;        // n_pad (FP64 mode)
    double4 *bcentre;       // n_blocks: block box centre (x,y,z, 0)
    double4 *bhalf;         // n_blocks: half extent
    double4 *scentre, *shalf; // n_super: super-block boxes
    double *alpha_s;        // n_pad (0 for phantoms)
    double *inv_alpha_s;    // n_pad (0 for phantoms)
    // block-pair list
    uint32_t *row_count;    // n_blocks + 1
    uint32_t *row_start;    // n_blocks + 1
    int2 *pairs;            // cap_tiles
    // per-evaluation data
    double *acc;            // 3 * n_pad (SoA x|y|z), FP64 accumulators
    float4 *mu32;           // n_pad
    double4 *mu64;          // n_pad
    float4 *mp32;           // 3 * n_pad: (q,dx,dy,dz) (Qxx,Qxy,Qxz,Qyy) (Qyz,Qzz,group,0)
    double4 *mp64;          // 3 * n_pad
    // PCG vectors, sorted order, SoA 3 * n_pad each
    double *vE, *vmu, *vr, *vp, *vq;
    double *partials;       // 3 sets (rz, pq, energy) of 2 * part_cap block partials
    int part_cap;           // >= the largest grid of any reducing kernel (n_blocks + MAX_PARTIALS)
    double *h_scalars;      // pinned host scratch (8 doubles) for scalar read-backs
    double *h_ring, *d_ring; // mapped pinned ring: |r|^2 of each PCG iteration, written by the device
    // ATOM lists: far class (atom_pairs.cu atom_far_setup)
    bool far_on;            // false: FP64 mode or beta = 0, every pair takes the full formula
    double far_x0;          // a pair is FAR iff x = R^3 w_i w_j >= far_x0 and R >= far_rmin
    double far_rmin;
    float far_q[6];         // far fit of erfcx in t = 1/R
    float4 *u32;            // n_pad: operand exchange of the persistent PCG kernel (atom_solve.cu)
    uint4 *tstore;          // TKHP_SOLVER_STORED_T: (G1, G2/3) of every list slot, [block][row][lane][8] float2 (atom_stored.cu)
    bool stored_t;          // the stored product is in use (flag set, MIXED/FIXED, ATOM lists requested)
    bool tstore_valid;      // tstore holds the elements of the current list
    bool fixed;             // TKHP_FIXED: int64 fixed-point accumulators in the FP32 pair kernels and the energy
    bool coop_ok;           // the device supports cooperative launches
    bool no_persist, no_fused_step;   // tkhp_params.solver_flags
    bool test_barrier_fault;          // TKHP_SOLVER_TEST_BARRIER_FAULT (tests: one CTA of the persistent kernels is lost)
    long long n_barrier_timeouts;     // persistent solves given up on a broken grid barrier and repeated on the fall-back path
    bool fuse_q;            // ATOM-mode T.mu kernel also forms q = p/alpha - T p - self p and p.q (PCG)
    int spec_iter;          // >= 0: the pair kernel about to be launched belongs to PCG iteration spec_iter
    DeviceState *h_state;   // pinned host copy of *st (list header), valid when header_valid
    bool header_valid;
    // host-entry staging (tkhp_polarize_host)
    double *h_pos, *h_alpha, *h_charge, *h_dipole, *h_quad, *h_field, *h_mu, *h_energy;
    cudaStream_t copy_stream;   // tkhp_polarize_host: the multipole H2D copies run beside the list build
    // list build: two branches beside the critical path (sort -> gather -> finer lists): [0] copies of the
    // inputs and the polarization-group sort, [1] the prescribed block-pair search (the finer lists do not
    // read it).  Forked and joined with events, also inside the captured graph.
    cudaStream_t side[2];
    cudaEvent_t fork_ev[2], join_ev[2];
    cudaEvent_t copy_ev[2];
    int32_t *h_group;
    // CLUSTER mode lists (see cluster.cu)
    void *cl_ws;
    size_t cl_ws_bytes;

    // CUDA graphs of one whole list build (about 30 small kernels, memsets and copies: launch bound).
    // A graph holds the three input pointers it was captured with; an MD integrator usually alternates
    // between two or three position buffers, so the last BUILD_GRAPH_SLOTS pointer triples keep their
    // graphs (least recently used slot is re-captured).
    static constexpr int BUILD_GRAPH_SLOTS = 4;
    struct BuildGraphSlot {
        cudaGraphExec_t exec;
        const void *key[3];             // d_pos, d_polarizability, d_group_id the graph was captured with
        long long launches;             // kernels inside the graph
        unsigned long long used;        // value of build_clock at the last replay (0: never)
    } build_slot[BUILD_GRAPH_SLOTS];
    unsigned long long build_clock;
    bool no_graph;                      // capture failed once: plain launches from then on
    long long n_graph_captures;         // graphs captured and instantiated since tkhp_create
    long long n_graph_replays;          // builds that ran as a graph replay
    long long n_plain_builds;           // builds enqueued as plain launches (stream 0, caller capturing, no_graph)

    cudaEvent_t ev[10];
    double last_ms[5];
    // launch accounting / live kernel timing (tkhp_profile_*)
    long long n_launches;               // kernels launched since the last reset
    bool prof;                          // record an event pair around every T.mu / field pair kernel
    int prof_n[3];                      // [0] T.mu launches, [1] field launches, [2] persistent solve kernels recorded
    cudaEvent_t prof_ev[3][2 * 64];
    int prof_iter[3][64];               // PCG iteration the recorded launch belongs to (-1: unconditional)
    bool prof_skip[3][64];              // the launch was a speculative no-op (iteration after convergence)
    long long prof_solve_matvecs;       // T.mu products done inside the recorded persistent solve kernels
    long long n_noop_launches;          // launches that returned at once for the same reason
};
constexpr int PROF_MAX = 64;
constexpr int RING = 16;          // slots of the PCG residual ring
constexpr int PCG_LAG = 2;        // iterations the host enqueues ahead of the last residual it has seen

// Bump allocator over the caller's workspace; with base == nullptr it only measures.
struct Carver {
    char *base;
    size_t off = 0;
    explicit Carver(void *b) : base(static_cast<char *>(b)) {}
    template <typename T>
    T *take(size_t count) {
        off = (off + 255) & ~size_t(255);
        T *p = base ? reinterpret_cast<T *>(base + off) : nullptr;
        off += count * sizeof(T);
        return p;
    }
};

inline int set_err(Ctx *c, int code, const char *fmt, const char *a = "") {
    if (c) snprintf(c->err, sizeof(c->err), fmt, a);
    return code;
}

#define TKHP_CUDA(ctx, call)                                                          \
    do {                                                                              \
        cudaError_t e_ = (call);                                                      \
        if (e_ != cudaSuccess) {                                                      \
            snprintf((ctx)->err, sizeof((ctx)->err), "%s:%d %s: %s", __FILE__, __LINE__, #call, \
                     cudaGetErrorString(e_));                                         \
            return TKHP_ECUDA;                                                        \
        }                                                                             \
    } while (0)

inline int div_up(long long a, long long b) { return (int)((a + b - 1) / b); }

// ---- host-side launchers implemented in the other translation units ----
int nblist_build(Ctx *c, const double *d_pos, const double *d_alpha, const int32_t *d_group,
                 cudaStream_t s);
int nblist_join(Ctx *c, cudaStream_t s);            // the caller's stream waits for the two side branches of nblist_build
int nblist_count_pairs(Ctx *c, cudaStream_t s);
int tiles_tmatvec(Ctx *c, cudaStream_t s);          // acc = T_real * (mu32|mu64), sorted space
int tiles_field(Ctx *c, cudaStream_t s);            // acc = unmasked inter-group field
size_t cluster_workspace_bytes(const tkhp_params *p, int n_blocks);
int cluster_build(Ctx *c, cudaStream_t s);
int cluster_init(Ctx *c);
int cluster_tmatvec(Ctx *c, cudaStream_t s);
int cluster_field(Ctx *c, cudaStream_t s);
long long cluster_slots(Ctx *c);
int atom_build(Ctx *c, cudaStream_t s);
void atom_far_setup(Ctx *c);
int atom_lists_configure(Ctx *c);
int atom_pairs_configure(Ctx *c);
int cluster_pairs_configure(Ctx *c);
int atom_solve_configure(Ctx *c);
bool atom_solve_eligible(Ctx *c);
bool tiles_solve_eligible(Ctx *c);
int tiles_solve_launch(Ctx *c, const double *d_field, double *d_mu, int use_guess, double tol, int max_iter, cudaStream_t s);
int atom_solve_launch(Ctx *c, const double *d_field, double *d_mu, int use_guess, double tol, int max_iter, cudaStream_t s);
int atom_tmatvec(Ctx *c, cudaStream_t s);
size_t atom_stored_bytes(const tkhp_params *p, int n_blocks);
int atom_stored_configure(Ctx *c);
int atom_stored_tmatvec(Ctx *c, cudaStream_t s);
int atom_field(Ctx *c, cudaStream_t s);
long long atom_slots(Ctx *c);

int run_tmatvec(Ctx *c, cudaStream_t s);            // dispatch on list mode; zeroes acc first
int run_field(Ctx *c, cudaStream_t s);
int do_perm_field(Ctx *c, const double *d_q, const double *d_dip, const double *d_quad, double *d_field,
                  cudaStream_t s);
int do_tmatvec(Ctx *c, const double *d_mu, double *d_out, cudaStream_t s);
int do_polar_solve(Ctx *c, const double *d_field, double *d_mu, double tol, int max_iter, int use_guess,
                   int *h_iters, double *h_rms, cudaStream_t s);
int do_polar_energy(Ctx *c, const double *d_mu, const double *d_field, double *d_energy, cudaStream_t s);
int ensure_header(Ctx *c, cudaStream_t s);          // list header on the host (one small sync per build)

// ---- fixed-point containers (TKHP_FIXED; eqs 2-3): a = int(round(x 2^fB)), x = real(a) / 2^fB.
// A 64-bit accumulator register is declared double in the kernels; in FIXED mode it carries the BITS
// of the int64 container (0.0 is integer 0), so that one kernel serves both modes.
constexpr int FIX_VEC_BITS = 34;      // field and T.mu accumulators
constexpr int FIX_ENERGY_BITS = 30;   // energy
__device__ __forceinline__ long long to_fixed(float x, int fb) { return __float2ll_rn(x * (float)(1ll << fb)); }
__device__ __forceinline__ void acc_add(double &a, float x, bool fixed) {
    if (fixed) a = __longlong_as_double(__double_as_longlong(a) + to_fixed(x, FIX_VEC_BITS));
    else a += (double)x;
}
__device__ __forceinline__ void acc_add(double &a, double x, bool) { a += x; }     // FP64 mode
__device__ __forceinline__ double acc_value(double a, bool fixed) {
    return fixed ? (double)__double_as_longlong(a) * (1.0 / (double)(1ll << FIX_VEC_BITS)) : a;
}

// warp helpers
__device__ __forceinline__ double warp_min(double v) {
    for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ double warp_max(double v) {
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ double warp_sum(double v) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

}  // namespace tkhp
