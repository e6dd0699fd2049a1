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
        const int I = IJ.x, J = IJ.y;
        const vec4 pi = xyzw[I * BLOCK + lane];
        const vec4 mi = mu[I * BLOCK + lane];
        real sx, sy, sz;
        tile_shift<real>(bcentre[I], bcentre[J], box, sx, sy, sz);
        const real xi = pi.x + sx, yi = pi.y + sy, zi = pi.z + sz;
        __syncwarp();
        s_pos[w][lane] = xyzw[J * BLOCK + lane];
        s_mu[w][lane] = mu[J * BLOCK + lane];
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

}  // namespace tkhp
