// tiles.cu -- TILES list mode: one warp per 32x32 block pair of the block-pair list.
//
// Paper: "a specific group of atoms interacts with another one in a block-matrix pattern ...
// load the parameters of the group of atoms and the output structures ... inside cache memory
// and/or registers ... CUDA built-in intrinsics can be used to read data from neighbor threads
// ... B_comp = B_size^2 computations without a single access to global memory" (P:L296-300,
// Fig. 11).  BASELINE.json north_star: "each warp handling one 32x32 block pair. The j-block is
// staged in shared memory or broadcast with __shfl_sync. Per-pair math runs in FP32 with FP64
// accumulation of fields, plus a full-FP64 variant."
//
// Mapping: lane l owns atom i = 32 I + l in registers; block J is staged once per tile in a
// per-warp shared-memory slab and read with the lane-rotated index (l + k) & 31 (conflict free);
// the partial result for atom j travels around the warp with the rotation (3 SHFL per step), so
// each unordered pair is evaluated once and both atoms are updated (Newton-pair symmetry, the
// "I <= J" half list of P:L335-366).  Tile partials are FP32 (MIXED) and are added to the FP64
// accumulators with one red.global.add.f64 per atom and tile (64-bit containers).
// Coordinates are block-local; the tile's image shift is computed once in FP64 from the block
// centres (exact when cutoff + 2 max_half < box/2, else the PPI variant wraps every pair).
#include "common.cuh"
#include "pair_math.cuh"
#include "reduce.cuh"

namespace tkhp {

constexpr int TILE_WARPS = 8;

template <typename real>
__device__ __forceinline__ real shfl_real(real v, int src) { return __shfl_sync(0xffffffffu, v, src); }

// minimum-image shift between two block centres, FP64 -> real
template <typename real>
__device__ __forceinline__ void tile_shift(const double4 &ci, const double4 &cj, double box, real &sx,
                                           real &sy, real &sz) {
    double dx = ci.x - cj.x, dy = ci.y - cj.y, dz = ci.z - cj.z;
    if (box > 0.0) {
        dx -= box * rint(dx / box);
        dy -= box * rint(dy / box);
        dz -= box * rint(dz / box);
    }
    sx = (real)dx; sy = (real)dy; sz = (real)dz;
}

template <typename real, bool PPI>
__device__ __forceinline__ void wrap_pair(real &Rx, real &Ry, real &Rz, const PairConsts<real> &k) {
    if (PPI) {
        Rx -= k.box * rint(Rx * k.inv_box);
        Ry -= k.box * rint(Ry * k.inv_box);
        Rz -= k.box * rint(Rz * k.inv_box);
    }
}

// a tile's contribution into the 64-bit accumulator of an atom: an FP64 atomic, or (TKHP_FIXED) an
// integer atomic on the int64 fixed-point container -- "we adopt a 64 bits container" with "atomic
// operations": the integer sum does not depend on the order of the tiles
template <typename real>
__device__ __forceinline__ void acc_atomic(double *p, real v, bool fixed) {
    if (fixed) atomicAdd(reinterpret_cast<unsigned long long *>(p), (unsigned long long)to_fixed((float)v, FIX_VEC_BITS));
    else atomicAdd(p, (double)v);
}

// the operand of T changes between the products of a persistent solve: read it through L2 (a plain or
// read-only load could hit a stale line of this SM's L1)
__device__ __forceinline__ float4 ld_operand(const float4 *p) { return __ldcg(p); }
__device__ __forceinline__ double4 ld_operand(const double4 *p) {
    const double2 a = __ldcg(reinterpret_cast<const double2 *>(p)), b = __ldcg(reinterpret_cast<const double2 *>(p) + 1);
    return make_double4(a.x, a.y, b.x, b.y);
}

// one tile (I, J) of the block-pair list, evaluated by one warp (lane = atom of block I)
template <typename real, bool PPI>
__device__ __forceinline__ void tile_tmu_one(const int2 IJ, typename Vec4<real>::type (*s_pos)[BLOCK],
                                             typename Vec4<real>::type (*s_mu)[BLOCK],
                                             const typename Vec4<real>::type *__restrict__ xyzw,
                                             const typename Vec4<real>::type *__restrict__ mu,
                                             const double4 *__restrict__ bcentre, double box, const PairConsts<real> &kc,
                                             double *__restrict__ acc, int n_pad, bool fixed) {
    using vec4 = typename Vec4<real>::type;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int I = IJ.x, J = IJ.y;
    const vec4 pi = xyzw[I * BLOCK + lane];
    const vec4 mi = ld_operand(mu + I * BLOCK + lane);
    real sx, sy, sz;
    tile_shift<real>(bcentre[I], bcentre[J], box, sx, sy, sz);
    const real xi = pi.x + sx, yi = pi.y + sy, zi = pi.z + sz;
    __syncwarp();
    s_pos[w][lane] = xyzw[J * BLOCK + lane];
    s_mu[w][lane] = ld_operand(mu + J * BLOCK + lane);
    __syncwarp();
    real ax = 0, ay = 0, az = 0;       // partial (T mu)_i
    real bx = 0, by = 0, bz = 0;       // travelling partial (T mu)_j
    if (I != J) {
#pragma unroll 4
        for (int k = 0; k < BLOCK; ++k) {
            const int jj = (lane + k) & 31;
            const vec4 pj = s_pos[w][jj];
            const vec4 mj = s_mu[w][jj];
            real Rx = xi - pj.x, Ry = yi - pj.y, Rz = zi - pj.z;
            wrap_pair<real, PPI>(Rx, Ry, Rz, kc);
            const real r2 = Rx * Rx + Ry * Ry + Rz * Rz;
            const real ww = pi.w * pj.w;
            const bool in = (r2 <= kc.rc2) && (ww > (real)0);
            real G[2];
            radial<2>(r2, ww, kc, G);
            const real m1 = in ? G[0] : (real)0, m2 = in ? G[1] : (real)0;
            tmu_apply<real>(m1, m2, Rx, Ry, Rz, mj.x, mj.y, mj.z, ax, ay, az);
            tmu_apply<real>(m1, m2, Rx, Ry, Rz, mi.x, mi.y, mi.z, bx, by, bz);
            const int src = (lane + 1) & 31;
            bx = shfl_real(bx, src); by = shfl_real(by, src); bz = shfl_real(bz, src);
        }
        const int sj = J * BLOCK + lane;
        acc_atomic(&acc[sj], bx, fixed);
        acc_atomic(&acc[n_pad + sj], by, fixed);
        acc_atomic(&acc[2 * n_pad + sj], bz, fixed);
    } else {
        // diagonal tile: every ordered pair i <- j, j != i (no mirror update)
#pragma unroll 4
        for (int k = 1; k < BLOCK; ++k) {
            const int jj = (lane + k) & 31;
            const vec4 pj = s_pos[w][jj];
            const vec4 mj = s_mu[w][jj];
            real Rx = xi - pj.x, Ry = yi - pj.y, Rz = zi - pj.z;
            wrap_pair<real, PPI>(Rx, Ry, Rz, kc);
            const real r2 = Rx * Rx + Ry * Ry + Rz * Rz;
            const real ww = pi.w * pj.w;
            const bool in = (r2 <= kc.rc2) && (ww > (real)0);
            real G[2];
            radial<2>(r2, ww, kc, G);
            const real m1 = in ? G[0] : (real)0, m2 = in ? G[1] : (real)0;
            tmu_apply<real>(m1, m2, Rx, Ry, Rz, mj.x, mj.y, mj.z, ax, ay, az);
        }
    }
    const int si = I * BLOCK + lane;
    acc_atomic(&acc[si], ax, fixed);
    acc_atomic(&acc[n_pad + si], ay, fixed);
    acc_atomic(&acc[2 * n_pad + si], az, fixed);
}

// ----------------------------------------------------------------------------- T.mu
template <typename real, bool PPI>
__global__ void __launch_bounds__(TILE_WARPS * 32)
k_tiles_tmu(const int2 *__restrict__ pairs, const DeviceState *__restrict__ st,
            const typename Vec4<real>::type *__restrict__ xyzw,
            const typename Vec4<real>::type *__restrict__ mu, const double4 *__restrict__ bcentre,
            double box, PairConsts<real> kc, double *__restrict__ acc, int n_pad, int iter) {
    using vec4 = typename Vec4<real>::type;
    __shared__ vec4 s_pos[TILE_WARPS][BLOCK];
    __shared__ vec4 s_mu[TILE_WARPS][BLOCK];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (iter >= 0 && iter >= st->conv_at) return;      // PCG already converged (pcg.cu)
    const bool fixed = sizeof(real) == 4 && kc.fixed != 0;
    const long long n_tiles = st->n_tiles;
    const long long stride = (long long)gridDim.x * TILE_WARPS;
    for (long long t = (long long)blockIdx.x * TILE_WARPS + w; t < n_tiles; t += stride) {
        const int2 IJ = pairs[t];
        tile_tmu_one<real, PPI>(IJ, s_pos, s_mu, xyzw, mu, bcentre, box, kc, acc, n_pad, fixed);
    }
}

// ----------------------------------------------------------------------------- permanent field
// Same-group pairs are skipped here and added by the FP64 correction pass (pcg.cu, k_field_finish):
// "compute ... then a separate scaling-correction pass".
template <typename real, bool PPI>
__global__ void __launch_bounds__(TILE_WARPS * 32)
k_tiles_field(const int2 *__restrict__ pairs, const DeviceState *__restrict__ st,
              const typename Vec4<real>::type *__restrict__ xyzw,
              const typename Vec4<real>::type *__restrict__ mp, const double4 *__restrict__ bcentre,
              double box, PairConsts<real> kc, double *__restrict__ acc, int n_pad, int iter) {
    using vec4 = typename Vec4<real>::type;
    __shared__ vec4 s_pos[TILE_WARPS][BLOCK];
    __shared__ vec4 s_mp[3][TILE_WARPS][BLOCK];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (iter >= 0 && iter >= st->conv_at) return;      // PCG already converged (pcg.cu)
    const bool fixed = sizeof(real) == 4 && kc.fixed != 0;
    const long long n_tiles = st->n_tiles;
    const long long stride = (long long)gridDim.x * TILE_WARPS;
    for (long long t = (long long)blockIdx.x * TILE_WARPS + w; t < n_tiles; t += stride) {
        const int2 IJ = pairs[t];
        const int I = IJ.x, J = IJ.y;
        const int si = I * BLOCK + lane, sj = J * BLOCK + lane;
        const vec4 pi = xyzw[si];
        const vec4 a0 = mp[si], a1 = mp[n_pad + si], a2 = mp[2 * n_pad + si];
        real sx, sy, sz;
        tile_shift<real>(bcentre[I], bcentre[J], box, sx, sy, sz);
        const real xi = pi.x + sx, yi = pi.y + sy, zi = pi.z + sz;
        __syncwarp();
        s_pos[w][lane] = xyzw[sj];
        s_mp[0][w][lane] = mp[sj];
        s_mp[1][w][lane] = mp[n_pad + sj];
        s_mp[2][w][lane] = mp[2 * n_pad + sj];
        __syncwarp();
        real ax = 0, ay = 0, az = 0, bx = 0, by = 0, bz = 0;
        const bool diag = (I == J);
#pragma unroll 2
        for (int k = diag ? 1 : 0; k < BLOCK; ++k) {
            const int jj = (lane + k) & 31;
            const vec4 pj = s_pos[w][jj];
            const vec4 b0 = s_mp[0][w][jj], b1 = s_mp[1][w][jj], b2 = s_mp[2][w][jj];
            real Rx = xi - pj.x, Ry = yi - pj.y, Rz = zi - pj.z;
            wrap_pair<real, PPI>(Rx, Ry, Rz, kc);
            const real r2 = Rx * Rx + Ry * Ry + Rz * Rz;
            const real ww = pi.w * pj.w;
            // group id travels in the z slot of the third multipole vector (exact in float up to 2^24,
            // compared as bit patterns for float; exact integers for double)
            const bool same = (a2.z == b2.z);
            const bool in = (r2 <= kc.rc2) && (ww > (real)0) && !same;
            real G[3];
            radial<3>(r2, ww, kc, G);
            if (!in) { G[0] = 0; G[1] = 0; G[2] = 0; }
            field_apply<real>(G, Rx, Ry, Rz, b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w, b2.x, b2.y,
                              ax, ay, az);
            if (!diag) {
                field_apply<real>(G, -Rx, -Ry, -Rz, a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w, a2.x,
                                  a2.y, bx, by, bz);
                const int src = (lane + 1) & 31;
                bx = shfl_real(bx, src); by = shfl_real(by, src); bz = shfl_real(bz, src);
            }
        }
        if (!diag) {
            acc_atomic(&acc[sj], bx, fixed);
            acc_atomic(&acc[n_pad + sj], by, fixed);
            acc_atomic(&acc[2 * n_pad + sj], bz, fixed);
        }
        acc_atomic(&acc[si], ax, fixed);
        acc_atomic(&acc[n_pad + si], ay, fixed);
        acc_atomic(&acc[2 * n_pad + si], az, fixed);
    }
}

// ----------------------------------------------------------------------------- persistent PCG (small systems)
// k_pcg_tiles: the whole PCG solve of a TILES-mode system as ONE cooperative kernel.  A box that is too
// small for the finer lists (config 0: 648 atoms, 230 tiles) is bound by launches: the launch-per-matvec
// path needs 3 launches and a host hand-shake per iteration (35 us per iteration for 5 us of work).
// Here the CTAs stay resident: per iteration the tiles (one warp each, grid-stride), then the vector
// work on one atom per thread (grid-stride) with the dot products as per-CTA partials that EVERY CTA
// adds in the same order after a grid barrier (reduce.cuh), four barriers per iteration.  The recurrences
// are those of pcg.cu (DESIGN.md section 2 "S"): the operand of T is the direction p rounded to the pair
// precision, the vectors are FP64.  Tile contributions are added with atomics (FP64: the sum depends on
// their order in the last bits, as in k_tiles_tmu; TKHP_FIXED: integer atomics, order-independent).
struct TilesSolveArgs {
    const int2 *pairs;
    const double4 *bcentre;
    const void *xyzw;          // float4 / double4, n_pad
    void *mu;                  // float4 / double4, n_pad: operand of T
    double *acc;               // 3 n_pad
    double *vE, *vmu, *vr, *vp, *vq;   // 3 n_pad each (SoA)
    const double *alpha_s, *inv_alpha_s;
    const int32_t *perm;
    const double *field;       // N x 3, caller's order
    double *mu_out;            // N x 3, caller's order: in (guess) / out
    double *part;              // 2 sets of 2 * gridDim.x partials
    volatile double *result;   // host-mapped: |r|^2, iterations, barrier time-out flag
    DeviceState *st;
    double box, tol, self;
    long long n_tiles;
    int n_pad, n_atoms, max_iter, use_guess;
    int test_fault;            // TKHP_SOLVER_TEST_BARRIER_FAULT: the last CTA never arrives at the first barrier
};

template <typename real, bool PPI>
__global__ void __launch_bounds__(TILE_WARPS * 32)
k_pcg_tiles(TilesSolveArgs a, PairConsts<real> kc) {
    using vec4 = typename Vec4<real>::type;
    __shared__ vec4 s_pos[TILE_WARPS][BLOCK];
    __shared__ vec4 s_mu[TILE_WARPS][BLOCK];
    const int w = threadIdx.x >> 5;
    const int n_pad = a.n_pad;
    const bool fixed = sizeof(real) == 4 && kc.fixed != 0;
    const vec4 *xyzw = static_cast<const vec4 *>(a.xyzw);
    vec4 *mu = static_cast<vec4 *>(a.mu);
    DeviceState *st = a.st;
    const int tid = blockIdx.x * blockDim.x + threadIdx.x, nthr = gridDim.x * blockDim.x;
    const long long wstride = (long long)gridDim.x * TILE_WARPS;
    double *part_a = a.part, *part_b = a.part + 2 * (size_t)gridDim.x;

    // mu0 = alpha E or the guess; E in sorted order; operand = mu0; accumulators cleared
    for (int s = tid; s < n_pad; s += nthr) {
        const int at = a.perm[s];
        const double al = a.alpha_s[s];
        double m[3] = {0, 0, 0};
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double e = at >= 0 ? a.field[3 * (size_t)at + c] : 0.0;
            m[c] = at >= 0 ? (a.use_guess ? a.mu_out[3 * (size_t)at + c] : al * e) : 0.0;
            a.vE[(size_t)c * n_pad + s] = e;
            a.vmu[(size_t)c * n_pad + s] = m[c];
            a.acc[(size_t)c * n_pad + s] = 0.0;
        }
        vec4 v; v.x = (real)m[0]; v.y = (real)m[1]; v.z = (real)m[2]; v.w = 0;
        mu[s] = v;
    }
    unsigned gen = 0;
    if (a.test_fault && blockIdx.x == gridDim.x - 1) return;   // tests: a CTA that is lost before the first barrier
    bool broken = !grid_barrier(st, gen);       // a barrier timed out: leave without touching the caller's mu
    double rz_old = 0.0, rr = 0.0;
    int it = 0;
    bool converged = false;
    for (int k = -1; k < a.max_iter && !broken; ++k) {
        // ---- acc = T v (v = mu0 or the direction)
        for (long long t = (long long)blockIdx.x * TILE_WARPS + w; t < a.n_tiles; t += wstride)
            tile_tmu_one<real, PPI>(a.pairs[t], s_pos, s_mu, xyzw, mu, a.bcentre, a.box, kc, a.acc, n_pad, fixed);
        if (!grid_barrier(st, gen)) { broken = true; break; }
        double s1 = 0.0, s2 = 0.0;
        if (k < 0) {
            // r = E - (mu/alpha - T mu - self mu); z = alpha r; p = z
            for (int s = tid; s < n_pad; s += nthr) {
                const double al = a.alpha_s[s], ia = a.inv_alpha_s[s];
                double p[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const size_t o = (size_t)c * n_pad + s;
                    const double m = a.vmu[o];
                    const double r = a.vE[o] - (m * ia - acc_value(__ldcg(a.acc + o), fixed) - a.self * m);
                    const double z = al * r;
                    a.vr[o] = r; a.vp[o] = z; p[c] = z;
                    a.acc[o] = 0.0;
                    s1 += r * z; s2 += r * r;
                }
                vec4 v; v.x = (real)p[0]; v.y = (real)p[1]; v.z = (real)p[2]; v.w = 0;
                mu[s] = v;
            }
            block_sum2(s1, s2);
            if (threadIdx.x == 0) { part_a[2 * blockIdx.x] = s1; part_a[2 * blockIdx.x + 1] = s2; }
            if (!grid_barrier(st, gen)) { broken = true; break; }
            grid_totals(part_a, rz_old, rr);
            if (sqrt(rr / a.n_atoms) < a.tol) { converged = true; break; }
            continue;
        }
        // ---- q = p/alpha - T p - self p ; p.q
        for (int s = tid; s < n_pad; s += nthr) {
            const double ia = a.inv_alpha_s[s];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const size_t o = (size_t)c * n_pad + s;
                const double p = a.vp[o];
                const double q = p * ia - acc_value(__ldcg(a.acc + o), fixed) - a.self * p;
                a.vq[o] = q;
                a.acc[o] = 0.0;
                s1 += p * q;
            }
        }
        block_sum2(s1, s2);
        if (threadIdx.x == 0) { part_b[2 * blockIdx.x] = s1; part_b[2 * blockIdx.x + 1] = 0.0; }
        if (!grid_barrier(st, gen)) { broken = true; break; }
        double pq, unused;
        grid_totals(part_b, pq, unused);
        const double gamma = rz_old / pq;
        // ---- mu += gamma p ; r -= gamma q ; (r.z, r.r)
        s1 = 0.0; s2 = 0.0;
        for (int s = tid; s < n_pad; s += nthr) {
            const double al = a.alpha_s[s];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const size_t o = (size_t)c * n_pad + s;
                a.vmu[o] += gamma * a.vp[o];
                const double r = a.vr[o] - gamma * a.vq[o];
                a.vr[o] = r;
                s1 += r * (al * r); s2 += r * r;
            }
        }
        block_sum2(s1, s2);
        if (threadIdx.x == 0) { part_a[2 * blockIdx.x] = s1; part_a[2 * blockIdx.x + 1] = s2; }
        if (!grid_barrier(st, gen)) { broken = true; break; }
        double rz_new;
        grid_totals(part_a, rz_new, rr);
        it = k + 1;
        if (sqrt(rr / a.n_atoms) < a.tol) { converged = true; break; }
        const double delta = rz_new / rz_old;
        rz_old = rz_new;
        // ---- p = alpha r + delta p, operand = p
        for (int s = tid; s < n_pad; s += nthr) {
            const double al = a.alpha_s[s];
            double p[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const size_t o = (size_t)c * n_pad + s;
                p[c] = al * a.vr[o] + delta * a.vp[o];
                a.vp[o] = p[c];
            }
            vec4 v; v.x = (real)p[0]; v.y = (real)p[1]; v.z = (real)p[2]; v.w = 0;
            mu[s] = v;
        }
        if (!grid_barrier(st, gen)) { broken = true; break; }
    }
    // ---- result in the caller's order; scalars to host-mapped memory
    for (int s = tid; s < n_pad && !broken; s += nthr) {
        const int at = a.perm[s];
        if (at >= 0) {
#pragma unroll
            for (int c = 0; c < 3; ++c) a.mu_out[3 * (size_t)at + c] = a.vmu[(size_t)c * n_pad + s];
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        st->rr = rr;
        st->iters = it;
        st->conv_at = converged ? it : 0x7fffffff;
        a.result[0] = rr;
        a.result[1] = (double)it;
        a.result[2] = broken ? 1.0 : 0.0;
        __threadfence_system();
    }
}

// TKHP_FIXED: the tile kernels have added int64 fixed-point values into `acc` with integer atomics (the
// paper's FP mode: deterministic whatever the order); back to FP64 values in place
__global__ void k_fixed_to_double(double *__restrict__ acc, size_t n) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) acc[i] = acc_value(acc[i], true);
}

template <typename real>
static PairConsts<real> make_consts(const tkhp_params &p) {
    PairConsts<real> k = {};
    k.beta = (real)p.ewald_beta;
    k.c1 = (real)(2.0 / SQRT_PI);
    k.c23 = (real)(4.0 / (3.0 * SQRT_PI));
    k.rc2 = (real)(p.cutoff * p.cutoff);
    k.box = (real)(p.box > 0.0 ? p.box : 1.0);
    k.inv_box = (real)(p.box > 0.0 ? 1.0 / p.box : 0.0);
    k.fixed = (sizeof(real) == 4 && p.precision == TKHP_FIXED) ? 1 : 0;
    return k;
}

static int tile_grid(Ctx *c) {
    // grid sized in whole waves of the SM count (4 CTAs of 8 warps per SM) unless the list is shorter
    long long want = (c->n_tiles_host + TILE_WARPS - 1) / TILE_WARPS;
    long long full = (long long)c->sm_count * 4;
    if (want < 1) want = 1;
    return (int)(want < full ? want : full);
}

// The host knows the list header (ensure_header): exactly one variant is launched.
#define TKHP_LAUNCH_TILES(KERNEL, REAL, XYZW, DATA)                                                   \
    do {                                                                                              \
        auto k = make_consts<REAL>(p);                                                                \
        if (c->h_state->per_pair_image)                                                               \
            KERNEL<REAL, true><<<grid, TILE_WARPS * 32, 0, s>>>(c->pairs, c->st, XYZW, DATA, c->bcentre, \
                                                                p.box, k, c->acc, c->n_pad, c->spec_iter);          \
        else                                                                                          \
            KERNEL<REAL, false><<<grid, TILE_WARPS * 32, 0, s>>>(c->pairs, c->st, XYZW, DATA, c->bcentre, \
                                                                 p.box, k, c->acc, c->n_pad, c->spec_iter);         \
    } while (0)

int tiles_tmatvec(Ctx *c, cudaStream_t s) {
    const int grid = tile_grid(c);
    const tkhp_params &p = c->p;
    if (p.precision != TKHP_FP64)
        TKHP_LAUNCH_TILES(k_tiles_tmu, float, c->xyzw32, c->mu32);
    else
        TKHP_LAUNCH_TILES(k_tiles_tmu, double, c->xyzw64, c->mu64);
    c->n_launches += 1;
    if (c->fixed) {
        const size_t n3 = 3 * (size_t)c->n_pad;
        k_fixed_to_double<<<(unsigned)((n3 + 255) / 256), 256, 0, s>>>(c->acc, n3);
        c->n_launches += 1;
    }
    TKHP_CUDA(c, cudaGetLastError());
    return TKHP_OK;
}

int tiles_field(Ctx *c, cudaStream_t s) {
    const int grid = tile_grid(c);
    const tkhp_params &p = c->p;
    if (p.precision != TKHP_FP64)
        TKHP_LAUNCH_TILES(k_tiles_field, float, c->xyzw32, c->mp32);
    else
        TKHP_LAUNCH_TILES(k_tiles_field, double, c->xyzw64, c->mp64);
    c->n_launches += 1;
    if (c->fixed) {
        const size_t n3 = 3 * (size_t)c->n_pad;
        k_fixed_to_double<<<(unsigned)((n3 + 255) / 256), 256, 0, s>>>(c->acc, n3);
        c->n_launches += 1;
    }
    TKHP_CUDA(c, cudaGetLastError());
    return TKHP_OK;
}

// ---- host side of the persistent TILES solve
constexpr int TILES_SOLVE_MAX_PAD = 16384;      // larger systems amortise their launches

template <typename real, bool PPI>
static const void *tiles_solve_fn() { return (const void *)k_pcg_tiles<real, PPI>; }
static const void *tiles_solve_pick(Ctx *c) {
    const bool ppi = c->h_state->per_pair_image != 0;
    if (c->p.precision == TKHP_FP64) return ppi ? tiles_solve_fn<double, true>() : tiles_solve_fn<double, false>();
    return ppi ? tiles_solve_fn<float, true>() : tiles_solve_fn<float, false>();
}
static int tiles_solve_grid(Ctx *c) {
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, tiles_solve_pick(c), TILE_WARPS * 32, 0) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    long long want = (c->h_state->n_tiles + TILE_WARPS - 1) / TILE_WARPS;
    const long long atoms = (c->n_pad + TILE_WARPS * 32 - 1) / (TILE_WARPS * 32);
    if (want < atoms) want = atoms;
    const long long cap = (long long)per_sm * c->sm_count;
    if (want > cap) want = cap;
    if (want > c->part_cap) want = c->part_cap;
    return (int)(want < 1 ? 0 : want);
}

// (list header on the host: ensure_header has run)
bool tiles_solve_eligible(Ctx *c) {
    return c->coop_ok && !c->no_persist && c->list_mode_in_use == TKHP_LIST_TILES && c->n_pad <= TILES_SOLVE_MAX_PAD &&
           c->h_state->n_tiles > 0 && tiles_solve_grid(c) > 0;
}

int tiles_solve_launch(Ctx *c, const double *d_field, double *d_mu, int use_guess, double tol, int max_iter, cudaStream_t s) {
    const tkhp_params &p = c->p;
    const bool f64 = p.precision == TKHP_FP64;
    TilesSolveArgs a;
    a.pairs = c->pairs; a.bcentre = c->bcentre;
    a.xyzw = f64 ? (const void *)c->xyzw64 : (const void *)c->xyzw32;
    a.mu = f64 ? (void *)c->mu64 : (void *)c->mu32;
    a.acc = c->acc;
    a.vE = c->vE; a.vmu = c->vmu; a.vr = c->vr; a.vp = c->vp; a.vq = c->vq;
    a.alpha_s = c->alpha_s; a.inv_alpha_s = c->inv_alpha_s; a.perm = c->perm;
    a.field = d_field; a.mu_out = d_mu;
    a.part = c->partials;
    a.result = c->d_ring;
    a.st = c->st;
    a.box = p.box; a.tol = tol;
    a.self = 4.0 * p.ewald_beta * p.ewald_beta * p.ewald_beta / (3.0 * SQRT_PI);
    a.n_tiles = c->h_state->n_tiles;
    a.n_pad = c->n_pad; a.n_atoms = c->n; a.max_iter = max_iter; a.use_guess = use_guess;
    a.test_fault = c->test_barrier_fault ? 1 : 0;
    const int grid = tiles_solve_grid(c);
    TKHP_CUDA(c, cudaMemsetAsync(&c->st->bar_count, 0, 2 * sizeof(unsigned), s));
    cudaError_t e;
    if (f64) {
        PairConsts<double> k = make_consts<double>(p);
        void *args[] = {&a, &k};
        e = cudaLaunchCooperativeKernel(tiles_solve_pick(c), dim3(grid), dim3(TILE_WARPS * 32), args, 0, s);
    } else {
        PairConsts<float> k = make_consts<float>(p);
        void *args[] = {&a, &k};
        e = cudaLaunchCooperativeKernel(tiles_solve_pick(c), dim3(grid), dim3(TILE_WARPS * 32), args, 0, s);
    }
    if (e != cudaSuccess) return set_err(c, TKHP_ECUDA, "cooperative launch of the persistent PCG kernel was refused%s");
    c->n_launches += 1;
    return TKHP_OK;
}

}  // namespace tkhp
