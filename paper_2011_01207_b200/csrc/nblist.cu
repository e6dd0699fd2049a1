// nblist.cu -- tkhp_nblist_build: spatial sort into 32-atom blocks and the block-pair list.
//
// Paper: cells with a 1-D numbering, atoms sorted by cell number, consecutive runs of
// B_size = 32 atoms form a group, group-pair adjacency -> compact list, phantom
// atoms pad the tail.  BASELINE.json north_star prescribes the bounding-box criterion
// "block pairs are kept by bounding-box distance against the cutoff plus a skin".
// Exact arithmetic of the key, the wrap and the box test: DESIGN.md section 3 (must be
// bit-reproducible, so every FP64 operation that matters uses __d*_rn: no FMA contraction).
//
// B200 mapping: counting sort on the Hilbert cell key (histogram with atomics, exclusive scan,
// scatter, in-cell rank by original index => deterministic and stable), one warp per 32-atom
// block for the gather + box reduction, one warp per block row for a two-level (32-block
// super-box, then block) pair search, two passes (count, fill) around a device scan.  All of it
// is HBM/latency bound and runs without a host synchronisation.
#include "common.cuh"

namespace tkhp {

// ----------------------------------------------------------------------------- scan
constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 8;                       // per thread
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;  // 2048

__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t *total) {
    __shared__ uint32_t warp_sums[SCAN_THREADS / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    uint32_t x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
    }
    if (lane == 31) warp_sums[wid] = x;
    __syncthreads();
    if (wid == 0) {
        uint32_t s = lane < SCAN_THREADS / 32 ? warp_sums[lane] : 0;
#pragma unroll
        for (int o = 1; o < SCAN_THREADS / 32; o <<= 1) {
            uint32_t y = __shfl_up_sync(0xffffffffu, s, o);
            if (lane >= o) s += y;
        }
        if (lane < SCAN_THREADS / 32) warp_sums[lane] = s;
    }
    __syncthreads();
    uint32_t base = wid ? warp_sums[wid - 1] : 0;
    *total = warp_sums[SCAN_THREADS / 32 - 1];
    __syncthreads();
    return base + x - v;
}

__global__ void k_scan_reduce(const uint32_t *__restrict__ in, uint32_t n, uint32_t *__restrict__ sums) {
    uint32_t base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
    uint32_t s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k)
        if (base + k < n) s += in[base + k];
    uint32_t total;
    block_exclusive_scan(s, &total);
    if (threadIdx.x == 0) sums[blockIdx.x] = total;
}

__global__ void k_scan_sums(uint32_t *sums, uint32_t n_blocks) {
    // single block: exclusive scan of the block sums, SCAN_THREADS at a time
    __shared__ uint32_t carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (uint32_t base = 0; base < n_blocks; base += SCAN_THREADS) {
        uint32_t i = base + threadIdx.x;
        uint32_t v = i < n_blocks ? sums[i] : 0;
        uint32_t total;
        uint32_t ex = block_exclusive_scan(v, &total);
        uint32_t c = carry;
        if (i < n_blocks) sums[i] = c + ex;
        __syncthreads();
        if (threadIdx.x == 0) carry = c + total;
        __syncthreads();
    }
}

__global__ void k_scan_apply(const uint32_t *__restrict__ in, uint32_t n,
                             const uint32_t *__restrict__ sums, uint32_t *__restrict__ out) {
    uint32_t base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
    uint32_t v[SCAN_ITEMS];
    uint32_t s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        v[k] = base + k < n ? in[base + k] : 0;
        s += v[k];
    }
    uint32_t total;
    uint32_t ex = block_exclusive_scan(s, &total) + sums[blockIdx.x];
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        if (base + k < n) out[base + k] = ex;
        ex += v[k];
    }
}

// out[i] = sum_{k<i} in[k], i = 0..n-1 (so pass n = bins + 1 to get the grand total at out[bins]).
static void exclusive_scan(Ctx *c, const uint32_t *in, uint32_t *out, uint32_t n, uint32_t *tmp, cudaStream_t s) {
    c->n_launches += 3;
    uint32_t nb = (n + SCAN_TILE - 1) / SCAN_TILE;
    k_scan_reduce<<<nb, SCAN_THREADS, 0, s>>>(in, n, tmp);
    k_scan_sums<<<1, SCAN_THREADS, 0, s>>>(tmp, nb);
    k_scan_apply<<<nb, SCAN_THREADS, 0, s>>>(in, n, tmp, out);
}

// ----------------------------------------------------------------------------- keys
// w = x - L floor(x/L), clamped into [0,L)  (Q16)
__device__ __forceinline__ double wrap_coord(double x, double box) {
    if (box <= 0.0) return x;
    double w = __dsub_rn(x, __dmul_rn(box, floor(__ddiv_rn(x, box))));
    if (w >= box) w = __dsub_rn(w, box);
    if (w < 0.0) w = 0.0;
    return w;
}

// Hilbert index of a cell on a 2^b grid (Skilling's transpose algorithm, own restatement):
// undo excess work from the top bit down, Gray-encode, then interleave bits x,y,z from the
// most significant bit.
__device__ __forceinline__ uint32_t hilbert3(uint32_t x, uint32_t y, uint32_t z, int b) {
    uint32_t X[3] = {x, y, z};
    const uint32_t M = 1u << (b - 1);
    for (uint32_t Q = M; Q > 1; Q >>= 1) {
        const uint32_t P = Q - 1;
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            if (X[i] & Q) {
                X[0] ^= P;
            } else {
                uint32_t t = (X[0] ^ X[i]) & P;
                X[0] ^= t;
                X[i] ^= t;
            }
        }
    }
    X[1] ^= X[0];
    X[2] ^= X[1];
    uint32_t t = 0;
    for (uint32_t Q = M; Q > 1; Q >>= 1)
        if (X[2] & Q) t ^= Q - 1;
    X[0] ^= t; X[1] ^= t; X[2] ^= t;
    uint32_t key = 0;
    for (int k = b - 1; k >= 0; --k) {
        key = (key << 1) | ((X[0] >> k) & 1u);
        key = (key << 1) | ((X[1] >> k) & 1u);
        key = (key << 1) | ((X[2] >> k) & 1u);
    }
    return key;
}

__global__ void k_state_init(DeviceState *st, int bits, double inv_h) {
    memset(st, 0, sizeof(DeviceState));
    st->grid_bits = bits;
    st->grid_inv_h = inv_h;
    for (int c = 0; c < 3; ++c) {
        st->lo[c] = INFINITY;
        st->hi[c] = -INFINITY;
    }
}

__device__ __forceinline__ void atomic_min_double(double *addr, double v) {
    unsigned long long *a = reinterpret_cast<unsigned long long *>(addr);
    unsigned long long old = *a;
    while (v < __longlong_as_double((long long)old)) {
        unsigned long long assumed = old;
        old = atomicCAS(a, assumed, (unsigned long long)__double_as_longlong(v));
        if (old == assumed) break;
    }
}
__device__ __forceinline__ void atomic_max_double(double *addr, double v) {
    unsigned long long *a = reinterpret_cast<unsigned long long *>(addr);
    unsigned long long old = *a;
    while (v > __longlong_as_double((long long)old)) {
        unsigned long long assumed = old;
        old = atomicCAS(a, assumed, (unsigned long long)__double_as_longlong(v));
        if (old == assumed) break;
    }
}

// open boundary only: bounding box of all atoms
__global__ void k_extent(const double *__restrict__ pos, int n, DeviceState *st) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    double lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    if (i < n) {
        for (int c = 0; c < 3; ++c) {
            double v = pos[3 * (size_t)i + c];
            if (isfinite(v)) { lo[c] = v; hi[c] = v; }
        }
    }
    for (int c = 0; c < 3; ++c) {
        double l = warp_min(lo[c]), h = warp_max(hi[c]);
        if ((threadIdx.x & 31) == 0) {
            atomic_min_double(&st->lo[c], l);
            atomic_max_double(&st->hi[c], h);
        }
    }
}

// open boundary only: extent = 1.000001 max_axis(hi-lo) + 1e-9 ; b = smallest 1..b_max with
// extent / 2^b <= 2.5, else b_max (= 6 for open boundaries) ; inv_h = 2^b / extent
__global__ void k_grid_from_extent(DeviceState *st, int b_max) {
    double span = 0.0;
    for (int c = 0; c < 3; ++c) {
        st->grid_origin[c] = st->lo[c];
        span = fmax(span, __dsub_rn(st->hi[c], st->lo[c]));
    }
    double extent = __dadd_rn(__dmul_rn(span, 1.000001), 1e-9);
    int b = 1;
    while (__ddiv_rn(extent, (double)(1 << b)) > 2.5 && b < b_max) ++b;      // coarser cells beyond b_max: only the sort locality suffers
    st->grid_bits = b;
    st->grid_inv_h = __ddiv_rn((double)(1 << b), extent);
}

__global__ void k_cell_keys(const double *__restrict__ pos, const double *__restrict__ alpha,
                            const int32_t *__restrict__ group, int n, double box,
                            DeviceState *st, uint32_t *__restrict__ key,
                            uint32_t *__restrict__ cell_count) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int b = st->grid_bits;
    const double inv_h = st->grid_inv_h;
    const uint32_t top = (1u << b) - 1u;
    uint32_t cell[3];
    bool ok = true;
    for (int c = 0; c < 3; ++c) {
        double x = pos[3 * (size_t)i + c];
        if (!isfinite(x)) { ok = false; x = 0.0; }
        double w = box > 0.0 ? wrap_coord(x, box) : __dsub_rn(x, st->grid_origin[c]);
        double f = floor(__dmul_rn(w, inv_h));
        long long ci = (long long)f;
        if (ci < 0) ci = 0;
        if (ci > (long long)top) ci = top;
        cell[c] = (uint32_t)ci;
    }
    if (!ok) st->err_nonfinite = 1;
    double a = alpha[i];
    if (!(a > 0.0) || !isfinite(a)) st->err_bad_alpha = 1;
    int g = group[i];
    if (g < 0 || g >= n) st->err_bad_group = 1;
    uint32_t k = ok ? hilbert3(cell[0], cell[1], cell[2], b) : 0u;
    key[i] = k;
    atomicAdd(&cell_count[k], 1u);
}

__global__ void k_group_keys(const int32_t *__restrict__ group, int n, uint32_t *__restrict__ key,
                             uint32_t *__restrict__ count) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int g = group[i];
    uint32_t k = (g < 0 || g >= n) ? 0u : (uint32_t)g;
    key[i] = k;
    atomicAdd(&count[k], 1u);
}

// unordered scatter into the bin's segment (count is consumed: counts down to zero)
__global__ void k_bin_scatter(const uint32_t *__restrict__ key, int n, const uint32_t *__restrict__ start,
                              uint32_t *__restrict__ count, int32_t *__restrict__ tmp_idx) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint32_t k = key[i];
    uint32_t slot = start[k] + (atomicSub(&count[k], 1u) - 1u);
    tmp_idx[slot] = i;
}

// deterministic order inside a bin: rank = number of members with a smaller original index
__global__ void k_bin_rank(const uint32_t *__restrict__ key, int n, const uint32_t *__restrict__ start,
                           const int32_t *__restrict__ tmp_idx, int32_t *__restrict__ out_idx) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint32_t k = key[i];
    uint32_t s = start[k], e = start[k + 1];
    uint32_t rank = 0;
    for (uint32_t t = s; t < e; ++t) rank += (tmp_idx[t] < i) ? 1u : 0u;
    out_idx[s + rank] = i;
}

__global__ void k_fill_i32(int32_t *p, int n, int32_t v) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}

// sort indices 0..n-1 by (key, index); start[0..n_bins] = bin offsets (kept for the groups)
static void counting_sort(Ctx *c, const uint32_t *key, int n, uint32_t n_bins, uint32_t *count, uint32_t *start,
                          uint32_t *scan_tmp, int32_t *tmp_idx, int32_t *out_idx, cudaStream_t s) {
    exclusive_scan(c, count, start, n_bins + 1, scan_tmp, s);
    c->n_launches += 2;
    int nb = div_up(n, 256);
    k_bin_scatter<<<nb, 256, 0, s>>>(key, n, start, count, tmp_idx);
    k_bin_rank<<<nb, 256, 0, s>>>(key, n, start, tmp_idx, out_idx);
}

// ----------------------------------------------------------------------------- gather + boxes
// One warp per block.  Box: lo/hi = exact min/max of the wrapped coordinates of the block's real
// atoms; centre = 0.5 (lo+hi), half = 0.5 (hi-lo).  Local coordinates = wrapped - centre (FP64
// subtraction, then one rounding to FP32): |local| <= half extent, so FP32 resolution is that of
// a few-Angstrom number whatever the box size (SURVEY hard part 2; paper's analogue: "distances
// in DP before casting").
__global__ void k_gather_blocks(const double *__restrict__ pos, const double *__restrict__ alpha,
                                const int32_t *__restrict__ perm, int n_blocks, double box, double thole_a,
                                int want64, float4 *__restrict__ xyzw32, double4 *__restrict__ xyzw64,
                                double4 *__restrict__ bcentre, double4 *__restrict__ bhalf,
                                double *__restrict__ alpha_s, double *__restrict__ inv_alpha_s,
                                DeviceState *st) {
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (warp >= n_blocks) return;
    const int slot = warp * BLOCK + lane;
    const int a = perm[slot];
    double w[3] = {0.0, 0.0, 0.0};
    double al = 0.0;
    if (a >= 0) {
        for (int c = 0; c < 3; ++c) w[c] = wrap_coord(pos[3 * (size_t)a + c], box);
        al = alpha[a];
    }
    double ctr[3], hf[3];
    for (int c = 0; c < 3; ++c) {
        double lo = warp_min(a >= 0 ? w[c] : INFINITY);
        double hi = warp_max(a >= 0 ? w[c] : -INFINITY);
        ctr[c] = __dmul_rn(0.5, __dadd_rn(lo, hi));
        hf[c] = __dmul_rn(0.5, __dsub_rn(hi, lo));
    }
    if (lane == 0) {
        bcentre[warp] = make_double4(ctr[0], ctr[1], ctr[2], 0.0);
        bhalf[warp] = make_double4(hf[0], hf[1], hf[2], 0.0);
        double hmax = fmax(hf[0], fmax(hf[1], hf[2]));
        atomicMax(&st->max_half_bits, (unsigned long long)__double_as_longlong(hmax));
    }
    double lx, ly, lz, wf;
    if (a >= 0) {
        lx = w[0] - ctr[0];
        ly = w[1] - ctr[1];
        lz = w[2] - ctr[2];
        wf = (al > 0.0) ? sqrt(thole_a / al) : 0.0;      // w = (a/alpha)^(1/2): a u^3 = R^3 w_i w_j
    } else {
        // phantom atoms: far away and mutually distant, so the cutoff test removes them
        lx = ly = lz = (double)PHANTOM_FAR * (double)(1 + lane);
        wf = 0.0;
    }
    xyzw32[slot] = make_float4((float)lx, (float)ly, (float)lz, (float)wf);
    if (want64) xyzw64[slot] = make_double4(lx, ly, lz, wf);
    alpha_s[slot] = a >= 0 ? al : 0.0;
    inv_alpha_s[slot] = (a >= 0 && al > 0.0) ? 1.0 / al : 0.0;
}

// conservative box of SUPER consecutive blocks (only used to generate candidates)
__global__ void k_super_boxes(const double4 *__restrict__ bcentre, const double4 *__restrict__ bhalf,
                              int n_blocks, int n_super, double4 *__restrict__ scentre,
                              double4 *__restrict__ shalf) {
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (warp >= n_super) return;
    const int b = warp * SUPER + lane;
    double lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    if (b < n_blocks) {
        double4 c = bcentre[b], h = bhalf[b];
        lo[0] = c.x - h.x; hi[0] = c.x + h.x;
        lo[1] = c.y - h.y; hi[1] = c.y + h.y;
        lo[2] = c.z - h.z; hi[2] = c.z + h.z;
    }
    double ctr[3], hf[3];
    for (int c = 0; c < 3; ++c) {
        double l = warp_min(lo[c]), h = warp_max(hi[c]);
        ctr[c] = 0.5 * (l + h);
        hf[c] = 0.5 * (h - l) * (1.0 + 1e-12) + 1e-9;   // inflate: candidates must be a superset
    }
    if (lane == 0) {
        scentre[warp] = make_double4(ctr[0], ctr[1], ctr[2], 0.0);
        shalf[warp] = make_double4(hf[0], hf[1], hf[2], 0.0);
    }
}

// gap^2 between two boxes, exactly as DESIGN.md section 3 / SURVEY Q16
__device__ __forceinline__ double box_gap2(const double4 &ci, const double4 &hi, const double4 &cj,
                                           const double4 &hj, double box) {
    double dx = fabs(__dsub_rn(ci.x, cj.x));
    double dy = fabs(__dsub_rn(ci.y, cj.y));
    double dz = fabs(__dsub_rn(ci.z, cj.z));
    if (box > 0.0) {
        double ex = __dsub_rn(box, dx), ey = __dsub_rn(box, dy), ez = __dsub_rn(box, dz);
        if (ex < dx) dx = ex;
        if (ey < dy) dy = ey;
        if (ez < dz) dz = ez;
    }
    double gx = __dsub_rn(dx, __dadd_rn(hi.x, hj.x));
    double gy = __dsub_rn(dy, __dadd_rn(hi.y, hj.y));
    double gz = __dsub_rn(dz, __dadd_rn(hi.z, hj.z));
    if (gx < 0.0) gx = 0.0;
    if (gy < 0.0) gy = 0.0;
    if (gz < 0.0) gz = 0.0;
    return __dadd_rn(__dadd_rn(__dmul_rn(gx, gx), __dmul_rn(gy, gy)), __dmul_rn(gz, gz));
}

// One warp per block row I.  Level 1: lanes test 32 super-blocks at a time (conservative).
// Level 2: for each surviving super-block the lanes test its 32 blocks J >= I exactly.
// FILL = false: count only; FILL = true: write (I,J) in increasing J at row_start[I].
template <bool FILL>
__global__ void k_pair_search(const double4 *__restrict__ bcentre, const double4 *__restrict__ bhalf,
                              const double4 *__restrict__ scentre, const double4 *__restrict__ shalf,
                              int n_blocks, int n_super, double box, double reach2, double reach2_super,
                              uint32_t *__restrict__ row_count, const uint32_t *__restrict__ row_start,
                              int2 *__restrict__ pairs, long long cap_tiles, DeviceState *st) {
    const int I = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (I >= n_blocks) return;
    const double4 ci = bcentre[I], hi = bhalf[I];
    uint32_t count = 0;
    const uint32_t base = FILL ? row_start[I] : 0u;
    for (int s0 = (I / SUPER) & ~31; s0 < n_super; s0 += 32) {
        const int sj = s0 + lane;
        bool cand = false;
        if (sj < n_super && sj >= I / SUPER)
            cand = box_gap2(ci, hi, scentre[sj], shalf[sj], box) <= reach2_super;
        uint32_t m = __ballot_sync(0xffffffffu, cand);
        while (m) {
            const int s = s0 + (__ffs(m) - 1);
            m &= m - 1;
            const int J = s * SUPER + lane;
            bool keep = false;
            if (J < n_blocks && J >= I)
                keep = box_gap2(ci, hi, bcentre[J], bhalf[J], box) <= reach2;
            const uint32_t km = __ballot_sync(0xffffffffu, keep);
            if (FILL && keep) {
                const long long w = (long long)base + count + __popc(km & ((1u << lane) - 1u));
                if (w < cap_tiles) pairs[w] = make_int2(I, J);
            }
            count += __popc(km);
        }
    }
    if (!FILL && lane == 0) row_count[I] = count;
}

__global__ void k_list_finish(DeviceState *st, const uint32_t *__restrict__ row_start, int n_blocks,
                              long long cap_tiles, double box, double cutoff) {
    long long t = row_start[n_blocks];
    st->n_tiles = t;
    st->n_diag_tiles = n_blocks;
    if (t > cap_tiles) st->err_capacity = 1;
    // One minimum-image shift per tile is exact iff cutoff + 2 max_half < box/2.
    double hmax = __longlong_as_double((long long)st->max_half_bits);
    st->per_pair_image = (box > 0.0 && !(cutoff + 2.0 * hmax < 0.5 * box)) ? 1 : 0;
}

// ----------------------------------------------------------------------------- statistics
// Useful pairs: unordered {i,j}, i != j, R^2 <= rc^2, R = minimum image of r_i - r_j, all FP64 with
// the oracle's operation order (no contraction) so that the count is bit-exact.
__global__ void k_count_pairs(const int2 *__restrict__ pairs, long long n_tiles,
                              const int32_t *__restrict__ perm, const double *__restrict__ pos,
                              double box, double rc2, unsigned long long *__restrict__ total) {
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (warp >= n_tiles) return;
    const int2 t = pairs[warp];
    const int ai = perm[t.x * BLOCK + lane];
    const int aj = perm[t.y * BLOCK + lane];
    double xi[3] = {0, 0, 0}, xj[3] = {0, 0, 0};
    if (ai >= 0) for (int c = 0; c < 3; ++c) xi[c] = pos[3 * (size_t)ai + c];
    if (aj >= 0) for (int c = 0; c < 3; ++c) xj[c] = pos[3 * (size_t)aj + c];
    unsigned int cnt = 0;
    for (int k = 0; k < 32; ++k) {
        const int src = (lane + k) & 31;
        const int bj = __shfl_sync(0xffffffffu, aj, src);
        double d[3];
        for (int c = 0; c < 3; ++c) {
            double xo = __shfl_sync(0xffffffffu, xj[c], src);
            d[c] = __dsub_rn(xi[c], xo);
            if (box > 0.0) d[c] = __dsub_rn(d[c], __dmul_rn(box, nearbyint(__ddiv_rn(d[c], box))));
        }
        double r2 = __dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2]));
        bool ok = ai >= 0 && bj >= 0 && r2 <= rc2;
        if (t.x == t.y) ok = ok && (lane < src);   // diagonal tile: each unordered pair once
        cnt += ok ? 1u : 0u;
    }
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    if (lane == 0 && cnt) atomicAdd(total, (unsigned long long)cnt);
}

// ----------------------------------------------------------------------------- host driver
int nblist_build(Ctx *c, const double *d_pos, const double *d_alpha, const int32_t *d_group,
                 cudaStream_t s) {
    const int n = c->n;
    const tkhp_params &p = c->p;
    const int nb256 = div_up(n, 256);
    c->header_valid = false;

    // grid parameters: periodic -> host; open -> device reduction
    if (p.box > 0.0) {
        const int b = c->grid_bits_host;
        k_state_init<<<1, 1, 0, s>>>(c->st, b, (double)(1 << b) / p.box);
        c->n_launches += 1;
    } else {
        k_state_init<<<1, 1, 0, s>>>(c->st, 1, 1.0);
        k_extent<<<nb256, 256, 0, s>>>(d_pos, n, c->st);
        int b_max = 0;
        while ((1 << (3 * (b_max + 1))) <= c->n_cells_alloc) ++b_max;
        k_grid_from_extent<<<1, 1, 0, s>>>(c->st, b_max);
        c->n_launches += 3;
    }
    // ---- branch 0 (beside the spatial sort): copies of the inputs in the caller's order, and the members
    // of every polarization group sorted by (group, index) for the mask correction (A6)
    {
        cudaStream_t b = c->side[0];
        TKHP_CUDA(c, cudaEventRecord(c->fork_ev[0], s));
        TKHP_CUDA(c, cudaStreamWaitEvent(b, c->fork_ev[0], 0));
        TKHP_CUDA(c, cudaMemcpyAsync(c->pos_o, d_pos, sizeof(double) * 3 * (size_t)n, cudaMemcpyDeviceToDevice, b));
        TKHP_CUDA(c, cudaMemcpyAsync(c->group_o, d_group, sizeof(int32_t) * (size_t)n, cudaMemcpyDeviceToDevice, b));
        TKHP_CUDA(c, cudaMemsetAsync(c->count2, 0, sizeof(uint32_t) * ((size_t)n + 1), b));
        k_group_keys<<<nb256, 256, 0, b>>>(d_group, n, c->key2, c->count2);
        counting_sort(c, c->key2, n, (uint32_t)n, c->count2, c->grp_start, c->scan_tmp2, c->tmp_idx2, c->grp_members, b);
        TKHP_CUDA(c, cudaEventRecord(c->join_ev[0], b));
    }
    TKHP_CUDA(c, cudaMemsetAsync(c->cell_count, 0, sizeof(uint32_t) * ((size_t)c->n_cells_alloc + 1), s));
    k_cell_keys<<<nb256, 256, 0, s>>>(d_pos, d_alpha, d_group, n, p.box, c->st, c->key, c->cell_count);
    counting_sort(c, c->key, n, (uint32_t)c->n_cells_alloc, c->cell_count, c->cell_start, c->scan_tmp,
                  c->tmp_idx, c->perm, s);
    if (c->n_pad > n) { k_fill_i32<<<1, 32, 0, s>>>(c->perm + n, c->n_pad - n, -1); c->n_launches += 1; }

    // gather + boxes
    const int warps_per_cta = 8;
    k_gather_blocks<<<div_up(c->n_blocks, warps_per_cta), warps_per_cta * 32, 0, s>>>(
        d_pos, d_alpha, c->perm, c->n_blocks, p.box, p.thole_a, p.precision == TKHP_FP64 ? 1 : 0,
        c->xyzw32, c->xyzw64, c->bcentre, c->bhalf, c->alpha_s, c->inv_alpha_s, c->st);
    k_super_boxes<<<div_up(c->n_super, warps_per_cta), warps_per_cta * 32, 0, s>>>(
        c->bcentre, c->bhalf, c->n_blocks, c->n_super, c->scentre, c->shalf);

    // ---- branch 1: the prescribed block-pair list (count, scan, fill).  The finer lists are built from the
    // boxes, not from this list, so it runs beside them; the main stream does not touch scan_tmp any more.
    cudaStream_t s_main = s;
    s = c->side[1];
    TKHP_CUDA(c, cudaEventRecord(c->fork_ev[1], s_main));
    TKHP_CUDA(c, cudaStreamWaitEvent(s, c->fork_ev[1], 0));
    const double reach = p.cutoff + p.skin;
    const double reach2 = reach * reach;
    const double reach_super = reach * (1.0 + 1e-12) + 1e-9;
    const double reach2_super = reach_super * reach_super;
    const int grid_rows = div_up(c->n_blocks, warps_per_cta);
    k_pair_search<false><<<grid_rows, warps_per_cta * 32, 0, s>>>(
        c->bcentre, c->bhalf, c->scentre, c->shalf, c->n_blocks, c->n_super, p.box, reach2, reach2_super,
        c->row_count, c->row_start, c->pairs, c->cap_tiles, c->st);
    TKHP_CUDA(c, cudaMemsetAsync(c->row_count + c->n_blocks, 0, sizeof(uint32_t), s));
    exclusive_scan(c, c->row_count, c->row_start, (uint32_t)c->n_blocks + 1, c->scan_tmp, s);
    k_pair_search<true><<<grid_rows, warps_per_cta * 32, 0, s>>>(
        c->bcentre, c->bhalf, c->scentre, c->shalf, c->n_blocks, c->n_super, p.box, reach2, reach2_super,
        c->row_count, c->row_start, c->pairs, c->cap_tiles, c->st);
    k_list_finish<<<1, 1, 0, s>>>(c->st, c->row_start, c->n_blocks, c->cap_tiles, p.box, p.cutoff);
    TKHP_CUDA(c, cudaEventRecord(c->join_ev[1], s));
    c->n_launches += 7;   // cell keys, group keys, gather, super boxes, 2 x pair search, finish
    TKHP_CUDA(c, cudaGetLastError());
    return TKHP_OK;
}

int nblist_join(Ctx *c, cudaStream_t s) {
    TKHP_CUDA(c, cudaStreamWaitEvent(s, c->join_ev[0], 0));
    TKHP_CUDA(c, cudaStreamWaitEvent(s, c->join_ev[1], 0));
    return TKHP_OK;
}

int nblist_count_pairs(Ctx *c, cudaStream_t s) {
    // needs n_tiles on the host: caller synchronised and filled n_tiles_host
    unsigned long long *total = reinterpret_cast<unsigned long long *>(&c->st->n_pairs_within_cutoff);
    TKHP_CUDA(c, cudaMemsetAsync(total, 0, sizeof(unsigned long long), s));
    if (c->n_tiles_host > 0) {
        const long long warps = c->n_tiles_host;
        k_count_pairs<<<div_up(warps, 8), 256, 0, s>>>(c->pairs, warps, c->perm, c->pos_o, c->p.box,
                                                       c->p.cutoff * c->p.cutoff, total);
    }
    return TKHP_OK;
}

}  // namespace tkhp
