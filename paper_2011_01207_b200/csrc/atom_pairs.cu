// atom_pairs.cu -- ATOM list mode: the pair kernels that walk the exact per-atom lists
// (atom_lists.cu builds them, cluster.cuh has the layout).
//
// Paper, "List filtering": filtered neighbour lists, padded with phantom atoms, at the
// price of "a loss of coalesced memory access pattern".  ATOM mode carries the filtering down to
// the single atom:
//  * every list entry is a pair with R^2 <= r_c^2 for the positions of the build, so the pair
//    kernels contain no cutoff test, no predicate and no select -- padding entries point at a dummy
//    record with zero payload;
//  * a CTA owns a group of <= 8 consecutive 32-atom blocks (one warp each) and stages the group's
//    neighbourhood ONCE per chunk in shared memory, already shifted into the group's frame (no
//    image arithmetic in the loop).  A lane owns one atom and only ever updates that atom: no
//    atomics, bit-reproducible results;
//  * entries are 16-bit BYTE OFFSETS into the staged chunk, 8 per lane and ROW (a coalesced 512-byte
//    row per warp); the loss of coalescing the paper notes becomes per-lane gathers from shared
//    memory, in an order that avoids bank conflicts (atom_lists.cu);
//  * a block's rows come in SEGMENTS of FAR rows followed by NEAR rows.  FAR pairs (Thole damping
//    below FP32 resolution, z = beta R inside the far fit) need no Thole exponential and no erfcx
//    argument mapping: G1 and G2 come from t = 1/R, e^{-z^2} and one degree-5 polynomial, 2 MUFU and
//    28 FMA-pipe cycles per pair instead of 4 and 40;
//  * the FP32 T.mu kernel (k_atom_tmu32) evaluates two list entries per lane and call as the two
//    halves of packed FP32 instructions (f32x2.cuh), loads each list row from L2 into registers two
//    rows before its use (RowStream in atom_tmu.cuh; the cp.async list ring of round 1 was measured and
//    removed), and keeps the staged records as (x, y, z, mu_z), (mu_x, mu_y)
//    and w: a far pair reads 24 bytes of shared memory;
//  * a group with fewer than 5 blocks gives every block to 2, 4 or 8 warps (interleaved list rows);
//  * FP32 partial sums are flushed into FP64 registers every 4 rows.
#include "cluster.cuh"
#include "atom_tmu.cuh"
#include "atom_epilogue.cuh"

namespace tkhp {

constexpr int MODE_TMU = 0, MODE_FIELD = 1;

// ---- partial sums of one lane (generic kernels), flushed into FP64 registers every 4 rows --------
template <typename real>
struct Partial {
    real x = 0, y = 0, z = 0;
    __device__ __forceinline__ void flush(double &dx, double &dy, double &dz, bool fixed) {
        acc_add(dx, x, fixed); acc_add(dy, y, fixed); acc_add(dz, z, fixed);
        x = 0; y = 0; z = 0;
    }
};
// ---- generic pair evaluation (FP32 field, FP64 T.mu and field): W entries of one lane ----------
//   MODE_TMU   (T1,T2): out_i += -m1 mu_j + m2 (mu_j.R) R            staged: pos+w, mu
//   MODE_FIELD (F1,F2): field at i from (q,d,Q)_j, same-group pairs contribute zero here (the FP64
//                       correction pass adds them, pcg.cu)            staged: pos+w, 3 multipole vec4
// One staged record (4 reals).  FP32: 16 bytes at base + off.  FP64: the record is kept as two 16-byte
// halves, (x, y) at base + off/2 and (z, w) at base + half + off/2 (half = 16 bytes x records per array),
// so that a quarter warp's LDS.128 of eight records with different indices mod 8 is one wavefront, as
// in FP32 (a 32-byte record at a 32-byte stride can never be: only every other bank group is used).
template <typename real> struct RecLoad;
template <> struct RecLoad<float> {
    static __device__ __forceinline__ float4 get(const unsigned char *base, int, unsigned off) {
        return *reinterpret_cast<const float4 *>(base + off);
    }
};
template <> struct RecLoad<double> {
    static __device__ __forceinline__ double4 get(const unsigned char *base, int half, unsigned off) {
        const double2 lo = *reinterpret_cast<const double2 *>(base + (off >> 1));
        const double2 hi = *reinterpret_cast<const double2 *>(base + half + (off >> 1));
        return make_double4(lo.x, lo.y, hi.x, hi.y);
    }
};

template <typename real, int MODE, int W, bool THOLE>
__device__ __forceinline__ void eval_pairs(const unsigned char *s_base, int pay_stride, const unsigned (&off)[W],
                                           const typename Vec4<real>::type &pi, real gi,
                                           const PairConsts<real> &kc, Partial<real> &A) {
    using vec4 = typename Vec4<real>::type;
    constexpr int NK = MODE == MODE_TMU ? 2 : 3;
    real &ax = A.x, &ay = A.y, &az = A.z;
    vec4 pj[W];
    real Rx[W], Ry[W], Rz[W], r2[W], ww[W], G[W][NK];
    const int half = pay_stride >> 1;
#pragma unroll
    for (int u = 0; u < W; ++u) pj[u] = RecLoad<real>::get(s_base, half, off[u]);
    if (MODE == MODE_TMU) {
        vec4 mj[W];
#pragma unroll
        for (int u = 0; u < W; ++u) mj[u] = RecLoad<real>::get(s_base + pay_stride, half, off[u]);
#pragma unroll
        for (int u = 0; u < W; ++u) {
            Rx[u] = pi.x - pj[u].x; Ry[u] = pi.y - pj[u].y; Rz[u] = pi.z - pj[u].z;
            r2[u] = Rx[u] * Rx[u] + Ry[u] * Ry[u] + Rz[u] * Rz[u];
            ww[u] = pi.w * pj[u].w;
        }
        radial_w<NK, W, THOLE>(r2, ww, kc, G);
#pragma unroll
        for (int u = 0; u < W; ++u)
            tmu_apply<real>(G[u][0], G[u][1], Rx[u], Ry[u], Rz[u], mj[u].x, mj[u].y, mj[u].z, ax, ay, az);
    } else {
        vec4 b0v[W], b1v[W], b2v[W];
        bool in[W];
#pragma unroll
        for (int u = 0; u < W; ++u) {
            b0v[u] = RecLoad<real>::get(s_base + pay_stride, half, off[u]);
            b1v[u] = RecLoad<real>::get(s_base + 2 * pay_stride, half, off[u]);
            b2v[u] = RecLoad<real>::get(s_base + 3 * pay_stride, half, off[u]);
        }
#pragma unroll
        for (int u = 0; u < W; ++u) {
            Rx[u] = pi.x - pj[u].x; Ry[u] = pi.y - pj[u].y; Rz[u] = pi.z - pj[u].z;
            r2[u] = Rx[u] * Rx[u] + Ry[u] * Ry[u] + Rz[u] * Rz[u];
            ww[u] = pi.w * pj[u].w;
            in[u] = b2v[u].z != gi;
        }
        radial_w<NK, W, THOLE>(r2, ww, kc, G);
#pragma unroll
        for (int u = 0; u < W; ++u) {
            if (!in[u]) { G[u][0] = 0; G[u][1] = 0; G[u][2] = 0; }
            field_apply<real>(G[u], Rx[u], Ry[u], Rz[u], b0v[u].x, b0v[u].y, b0v[u].z, b0v[u].w, b1v[u].x,
                              b1v[u].y, b1v[u].z, b1v[u].w, b2v[u].x, b2v[u].y, ax, ay, az);
        }
    }
}

__device__ __forceinline__ void cp_async16(unsigned dst, const void *src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
// one record into local index l of an array region: FP32 16 bytes at l x 16; FP64 two halves (RecLoad)
template <int BYTES>
__device__ __forceinline__ void cp_async_rec(unsigned char *arr, int half, int l, const void *src) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(arr) + 16u * (unsigned)l;
    cp_async16(d, src);
    if (BYTES == 32) cp_async16(d + (unsigned)half, reinterpret_cast<const unsigned char *>(src) + 16);
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ uint4 lds128(unsigned addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
    return v;
}

// resident CTAs per SM the register allocation must allow: FP32 field 2 (112 KB of staging), FP64 T.mu 3
// (80 registers, 53 KB), FP64 field 1 (106 KB)
template <typename real, int MODE> struct MinCtas { static constexpr int N = (sizeof(real) == 8 && MODE == MODE_FIELD) ? 1 : (sizeof(real) == 8 ? 3 : 2); };

// ----------------------------------------------------------------------------- generic kernel
template <typename real, int MODE>
__global__ void __launch_bounds__(GT, MinCtas<real, MODE>::N)
k_atom_pairs(ClusterWs ws, const typename Vec4<real>::type *__restrict__ gpos,
             const typename Vec4<real>::type *__restrict__ stage_pos,
             const typename Vec4<real>::type *__restrict__ data,   // mu (n_pad) or multipoles (3 n_pad)
             PairConsts<real> kc, double *__restrict__ acc, int n_pad, int s_chunk,
             DeviceState *st, int iter, PcgFuse fuse) {
    if (iter >= 0 && iter >= st->conv_at) return;      // PCG already converged (pcg.cu)
    using vec4 = typename Vec4<real>::type;
    constexpr int NPAY = MODE == MODE_TMU ? 1 : 3;
    constexpr int SU = sizeof(real) == 8 ? 4 : 8;   // staged records in flight per thread
    extern __shared__ __align__(16) unsigned char smem_raw[];
    vec4 *s_pos = reinterpret_cast<vec4 *>(smem_raw);          // [s_chunk + N_DUMMY]; the dummies follow the group's largest chunk
    vec4 *s_pay = s_pos + (s_chunk + N_DUMMY);                 // NPAY arrays of [s_chunk + N_DUMMY]
    const int pstride = s_chunk + N_DUMMY;
    const int pay_stride = pstride * (int)sizeof(vec4);

    const int g = blockIdx.x, t = threadIdx.x, lane = t & 31, w = t >> 5;
    const int b0 = ws.group_first[g], nb = ws.group_first[g + 1] - b0;
    const int count = ws.stage_count[g];
    const int n_chunks = atom_chunks_of(count, s_chunk);
    const size_t gbase = (size_t)g * ws.s_cap;
    const int wpb = warps_per_block(nb);
    const int kb = w / wpb, part = w - kb * wpb;
    const bool active = kb < nb;
    const int blk = b0 + (active ? kb : 0);
    const int slot = blk * BLOCK + lane;
    const vec4 pi = gpos[slot];
    real gi = 0;
    if (MODE == MODE_FIELD) gi = data[2 * (size_t)n_pad + slot].z;
    const uint4 *__restrict__ rows = reinterpret_cast<const uint4 *>(ws.alist + (size_t)blk * ws.a_cap * 32) + lane;
    const int2 *__restrict__ seg = ws.aseg + (size_t)blk * NSEG_MAX;
    const int rows_last = (ws.a_cap >> 3) - 1;

    double dx = 0.0, dy = 0.0, dz = 0.0;
    Partial<real> A;
    int since_flush = 0;
    const bool fixed = sizeof(real) == 4 && kc.fixed != 0;

    if (t < N_DUMMY) {                         // permanent dummy records: far away, zero payload
        vec4 far, zero;
        far.x = far.y = far.z = (real)(-2.0f * PHANTOM_FAR); far.w = 0;
        zero.x = zero.y = zero.z = zero.w = 0;
        const int dmy = atom_dummy_index(count, n_chunks) + t;
        if (sizeof(real) == 4) {
            s_pos[dmy] = far;
            for (int k = 0; k < NPAY; ++k) s_pay[k * pstride + dmy] = zero;
        } else {                               // two 16-byte halves per record
            real *lo = reinterpret_cast<real *>(smem_raw + 16 * (size_t)dmy), *hi = reinterpret_cast<real *>(smem_raw + (pay_stride >> 1) + 16 * (size_t)dmy);
            lo[0] = far.x; lo[1] = far.y; hi[0] = far.z; hi[1] = far.w;
            for (int k = 0; k < NPAY; ++k) {
                real *plo = reinterpret_cast<real *>(smem_raw + (size_t)(k + 1) * pay_stride + 16 * (size_t)dmy);
                real *phi = reinterpret_cast<real *>(smem_raw + (size_t)(k + 1) * pay_stride + (pay_stride >> 1) + 16 * (size_t)dmy);
                plo[0] = 0; plo[1] = 0; phi[0] = 0; phi[1] = 0;
            }
        }
    }

    // My rows are part, part + wpb, ... of the block's row stream, whatever segment they fall in; a
    // row is loaded one whole row (8 pairs) before its use.  The loads are volatile asm so that they
    // stay where they are written.
    int d = 0;
    int2 sd = seg[0];
    int tg = part;                                   // my next row
    uint4 e_next = ldg_row(rows + (size_t)tg * 32);  // (the list area of a block has >= 8 rows)

    for (int c = 0; c < n_chunks; ++c) {
        __syncthreads();
        // staging of chunk c with cp.async (global -> shared without a register round trip): the
        // positions do not depend on the atom index, so a thread has its index loads and position
        // copies of up to SU records in flight together, then the payload copies by index.
        for (int l0 = t, i0 = c + t * n_chunks; i0 < count; l0 += SU * GT, i0 += SU * GT * n_chunks) {
            int a[SU];
#pragma unroll
            for (int u = 0; u < SU; ++u) {
                const int idx = i0 + u * GT * n_chunks;
                a[u] = idx < count ? ws.stage_atom[gbase + idx] : -1;
            }
#pragma unroll
            for (int u = 0; u < SU; ++u) {
                const int idx = i0 + u * GT * n_chunks;
                if (idx < count) cp_async_rec<sizeof(vec4)>(smem_raw, pay_stride >> 1, l0 + u * GT, stage_pos + gbase + idx);
            }
#pragma unroll
            for (int k = 0; k < NPAY; ++k) {
#pragma unroll
                for (int u = 0; u < SU; ++u)
                    if (a[u] >= 0) cp_async_rec<sizeof(vec4)>(smem_raw + (size_t)(k + 1) * pay_stride, pay_stride >> 1, l0 + u * GT, data + (size_t)k * n_pad + a[u]);
            }
        }
        cp_async_commit();
        cp_async_wait<0>();
        __syncthreads();
        if (!active) continue;
        const unsigned char *s_base = smem_raw;
        while (seg_chunk(sd) == c) {
            const int row0 = seg_row0(sd);
            const int nc[2] = {seg_far_calls(sd), seg_near_calls(sd)};
            const int r0[2] = {row0, row0 + ((nc[0] + 3) >> 2)};
#pragma unroll
            for (int cls = 0; cls < 2; ++cls) {
                const int rend = r0[cls] + ((nc[cls] + 3) >> 2);
                // the rows of one class; THOLE = false for FAR rows (the Thole term has died out)
                auto rows_of_class = [&](auto thole_tag) {
                    constexpr bool THOLE = decltype(thole_tag)::value;
                    for (; tg < rend; tg += wpb) {
                        const uint4 e = e_next;
                        e_next = ldg_row(rows + (size_t)min(tg + wpb, rows_last) * 32);
                        const int n_here = min(4, nc[cls] - 4 * (tg - r0[cls]));
                        const unsigned wd[4] = {e.x, e.y, e.z, e.w};
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            if (k < n_here) {
                                if (sizeof(real) == 8 && MODE == MODE_TMU) {       // FP64 T.mu: one pair at a time (registers: 3 CTAs per SM)
                                    const unsigned oa[1] = {wd[k] & 0xffffu}, ob[1] = {wd[k] >> 16};
                                    eval_pairs<real, MODE, 1, THOLE>(s_base, pay_stride, oa, pi, gi, kc, A);
                                    eval_pairs<real, MODE, 1, THOLE>(s_base, pay_stride, ob, pi, gi, kc, A);
                                } else {
                                    const unsigned o2[2] = {wd[k] & 0xffffu, wd[k] >> 16};
                                    eval_pairs<real, MODE, 2, THOLE>(s_base, pay_stride, o2, pi, gi, kc, A);
                                }
                            }
                        }
                        if (++since_flush == 4) {          // every 32 entries: FP32 partial -> 64-bit container
                            A.flush(dx, dy, dz, fixed);
                            since_flush = 0;
                        }
                    }
                };
                if (cls == 0 && kc.far_rows) rows_of_class(FalseTag());
                else rows_of_class(TrueTag());
            }
            sd = seg[++d];
        }
    }
    A.flush(dx, dy, dz, fixed);
    dx = acc_value(dx, fixed); dy = acc_value(dy, fixed); dz = acc_value(dz, fixed);
    pair_epilogue<MODE == MODE_TMU>(smem_raw, dx, dy, dz, wpb, part, active, slot, n_pad, acc, st, fuse);
}

// ----------------------------------------------------------------------------- FP32 T.mu kernel
// FAR: the far class is in use (MIXED, beta > 0); otherwise the first class of rows holds every pair
// and takes the full formula.  SPLIT: some group has < 5 blocks (small systems): every block of such
// a group is shared by 2, 4 or 8 warps; the host picks the instantiation for the whole grid.
template <bool FAR, bool SPLIT>
__global__ void __launch_bounds__(GT, 3)
k_atom_tmu32(ClusterWs ws, const float4 *__restrict__ gpos, const float4 *__restrict__ stage_pos,
             const float4 *__restrict__ mu, TmuConsts K, double *__restrict__ acc, int n_pad, int s_chunk,
             int rot_div, DeviceState *st, int iter, PcgFuse fuse) {
    if (iter >= 0 && iter >= st->conv_at) return;      // PCG already converged (pcg.cu)
    constexpr int SU = 4;                              // staged records in flight per thread
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int pstride = s_chunk + N_DUMMY;             // the dummy records follow the group's largest chunk
    float4 *s_a = reinterpret_cast<float4 *>(smem_raw);
    float2 *s_b = reinterpret_cast<float2 *>(smem_raw + (size_t)16 * pstride);
    float *s_w = reinterpret_cast<float *>(smem_raw + (size_t)24 * pstride);
    TmuSmem S;
    S.a = smem_raw; S.b = smem_raw + (size_t)16 * pstride; S.w = smem_raw + (size_t)24 * pstride;

    const int g = blockIdx.x, t = threadIdx.x, lane = t & 31, w = t >> 5;
    const int b0 = ws.group_first[g], nb = ws.group_first[g + 1] - b0;
    const int count = ws.stage_count[g];
    const int n_chunks = atom_chunks_of(count, s_chunk);
    const size_t gbase = (size_t)g * ws.s_cap;
    const int wpb = SPLIT ? warps_per_block(nb) : 1;
    // a group of 6 or 7 blocks leaves warps idle: which ones rotates with the wave the CTA belongs to
    // (g / SM count), so that the CTAs sharing an SM idle on different SM sub-partitions
    const int kb = SPLIT ? w / wpb : ((w + g / rot_div) & (GB - 1)), part = SPLIT ? w - kb * wpb : 0;
    const bool active = kb < nb;
    const int blk = b0 + (active ? kb : 0);
    const int slot = blk * BLOCK + lane;
    const int2 *__restrict__ seg = ws.aseg + (size_t)blk * NSEG_MAX;

    TmuLane L;
    {
        const float4 pi = gpos[slot];
        L.pxy = pk(pi.x, pi.y);
        L.nz = -pi.z;
        L.wl = pi.w * 1.4426950408889634f;
    }
    double dx = 0.0, dy = 0.0, dz = 0.0;
    PartialTmu A;

    if (t < N_DUMMY) {                         // permanent dummy records: far away, zero payload
        const float far = -2.0f * PHANTOM_FAR;
        const int dmy = atom_dummy_index(count, n_chunks) + t;
        s_a[dmy] = make_float4(far, far, far, 0.f);
        s_b[dmy] = make_float2(0.f, 0.f);
        s_w[dmy] = 0.f;
    }

    const int t_total = (active && n_chunks <= NCH_MAX) ? seg_row0(seg[NSEG_MAX - 1]) : 0;
    RowStream R;
    R.open(reinterpret_cast<const uint4 *>(ws.alist + (size_t)blk * ws.a_cap * 32) + lane, t_total, part, wpb);

    int d = 0, n_rows = 0;
    int2 sd = seg[0];
    int tg = part;                                   // my next row
    for (int c = 0; c < n_chunks; ++c) {
        __syncthreads();
        // staging of chunk c through registers: the records are re-packed on the way, (x, y, z, w) and
        // (mu_x, mu_y, mu_z, 0) in global memory become A, B and W; SU records per thread in flight
        for (int l0 = t, i0 = c + t * n_chunks; i0 < count; l0 += SU * GT, i0 += SU * GT * n_chunks) {
            int a[SU];
            float4 p[SU], m[SU];
#pragma unroll
            for (int u = 0; u < SU; ++u) {
                const int idx = i0 + u * GT * n_chunks;
                a[u] = idx < count ? ws.stage_atom[gbase + idx] : -1;
            }
#pragma unroll
            for (int u = 0; u < SU; ++u) {
                const int idx = i0 + u * GT * n_chunks;
                if (idx < count) p[u] = stage_pos[gbase + idx];
            }
#pragma unroll
            for (int u = 0; u < SU; ++u)
                if (a[u] >= 0) m[u] = __ldcg(mu + a[u]);
#pragma unroll
            for (int u = 0; u < SU; ++u) {
                if (a[u] >= 0) {
                    const int l = l0 + u * GT;
                    s_a[l] = make_float4(p[u].x, p[u].y, p[u].z, m[u].z);
                    s_b[l] = make_float2(m[u].x, m[u].y);
                    s_w[l] = p[u].w;
                }
            }
        }
        __syncthreads();
        if (!active) continue;
#ifdef TKHP_DBG_NOLOOP
        continue;
#endif
        tmu_walk<FAR>(seg, c, d, sd, tg, wpb, R, S, L, K, A, n_rows, dx, dy, dz);
    }
    A.flush(dx, dy, dz, K.fixed);
    dx = acc_value(dx, K.fixed != 0); dy = acc_value(dy, K.fixed != 0); dz = acc_value(dz, K.fixed != 0);
    pair_epilogue<true>(smem_raw, dx, dy, dz, wpb, part, active, slot, n_pad, acc, st, fuse);
}

// ----------------------------------------------------------------------------- host side
// Far-field fit (MIXED): erfcx(z) = s Q(s), s = 1/z, on z in [z_min, z_max], Q of degree 5 by
// interpolation at the Chebyshev nodes of [1/z_max, 1/z_min] (relative error of erfcx(z) + c z below
// 1e-7 for z_min = 1.3, z_max = 3.83).  Returned in t = 1/R: q_k = Q_k / beta^(k+1).
void atom_far_setup(Ctx *c) {
    const double beta = c->p.ewald_beta, rc = c->p.cutoff;
    const double z_min = 1.3, z_max = beta * rc * 1.002 + 1e-3;
    c->far_on = false;
    c->far_x0 = 0.0;
    c->far_rmin = 0.0;
    for (int k = 0; k < 6; ++k) c->far_q[k] = 0.f;
    // (FP64 with a Thole-free first class, x >= 45, was measured twice: T.mu 0.191 -> 0.213 ms and, with the 3-CTA kernel, 0.181 -> 0.190 ms on config 2; not used)
    if (c->p.precision == TKHP_FP64 || !(beta > 0.0) || z_max < 1.25 * z_min) return;    // no far class: full formula everywhere
    c->far_on = true;
    constexpr int D = 5;
    const double a = 1.0 / z_max, b = 1.0 / z_min;
    double x[D + 1], y[D + 1];
    for (int k = 0; k <= D; ++k) {
        x[k] = 0.5 * (a + b) + 0.5 * (b - a) * cos(3.14159265358979323846 * (k + 0.5) / (D + 1));
        const double z = 1.0 / x[k];
        y[k] = erfc(z) * exp(z * z) * z;                       // Q(s) = erfcx(1/s) / s
    }
    // Newton divided differences, then expansion to monomial coefficients
    double dd[D + 1];
    for (int k = 0; k <= D; ++k) dd[k] = y[k];
    for (int j = 1; j <= D; ++j)
        for (int k = D; k >= j; --k) dd[k] = (dd[k] - dd[k - 1]) / (x[k] - x[k - j]);
    double mono[D + 1] = {0};
    for (int k = D; k >= 0; --k) {                             // mono = mono * (s - x[k]) + dd[k]
        for (int i = D; i >= 1; --i) mono[i] = mono[i - 1] - x[k] * mono[i];
        mono[0] = -x[k] * mono[0] + dd[k];
    }
    double bp = beta;
    for (int k = 0; k <= D; ++k) { c->far_q[k] = (float)(mono[k] / bp); bp *= beta; }
    c->far_x0 = 20.0;                  // (1 + x) e^-x = 4e-8 at x = 20
    c->far_rmin = z_min / beta;
}

template <typename real, int MODE>
static int launch_atom_pairs(Ctx *c, const ClusterWs &ws, cudaStream_t s) {
    using vec4 = typename Vec4<real>::type;
    constexpr int NPAY = MODE == MODE_TMU ? 1 : 3;
    constexpr int which = sizeof(real) == 8;
    const int s_chunk = atom_chunk_capacity(which, ws.chunk_cap);
    const size_t smem = sizeof(vec4) * (size_t)(1 + NPAY) * (size_t)(s_chunk + N_DUMMY);
    PairConsts<real> k;
    k.beta = (real)c->p.ewald_beta;
    k.c1 = (real)(2.0 / SQRT_PI);
    k.c23 = (real)(4.0 / (3.0 * SQRT_PI));
    k.rc2 = (real)(c->p.cutoff * c->p.cutoff);
    k.box = (real)1;
    k.inv_box = (real)0;
    k.pb = k.nb2l = k.c1b = k.k3 = (real)0;
    k.fixed = c->fixed ? 1 : 0;
    k.far_rows = c->far_on ? 1 : 0;
    PcgFuse fuse;
    fuse.on = MODE == MODE_TMU && c->fuse_q;
    fuse.self = 4.0 * c->p.ewald_beta * c->p.ewald_beta * c->p.ewald_beta / (3.0 * SQRT_PI);
    fuse.vp = c->vp; fuse.inv_alpha = c->inv_alpha_s; fuse.vq = c->vq;
    fuse.part = c->partials + 2 * (size_t)c->part_cap;
    const vec4 *gpos = which ? (const vec4 *)ws.gpos64 : (const vec4 *)ws.gpos32;
    const vec4 *spos = which ? (const vec4 *)ws.stage_pos64 : (const vec4 *)ws.stage_pos32;
    const vec4 *data;
    if (MODE == MODE_TMU) data = which ? (const vec4 *)c->mu64 : (const vec4 *)c->mu32;
    else data = which ? (const vec4 *)c->mp64 : (const vec4 *)c->mp32;
    k_atom_pairs<real, MODE><<<ws.n_groups, GT, smem, s>>>(ws, gpos, spos, data, k, c->acc, c->n_pad, s_chunk, c->st, c->spec_iter, fuse);
    c->n_launches += 1;
    TKHP_CUDA(c, cudaGetLastError());
    return TKHP_OK;
}

static int launch_tmu32(Ctx *c, const ClusterWs &ws, cudaStream_t s) {
    const int s_chunk = atom_chunk_capacity(false, ws.chunk_cap);
    const double b = c->p.ewald_beta;
    TmuConsts K;
    K.pb = (float)((double)TKHP_ERFCX_P * b);
    K.nb2l = (float)(-1.4426950408889634 * b * b);
    K.c1b = (float)(2.0 / SQRT_PI * b);
    K.k3 = (float)(4.0 / (3.0 * SQRT_PI) * b * b * b);
    for (int k = 0; k < 6; ++k) K.q[k] = c->far_q[k];
    K.fixed = c->fixed ? 1 : 0;
    PcgFuse fuse;
    fuse.on = c->fuse_q;
    fuse.self = 4.0 * b * b * b / (3.0 * SQRT_PI);
    fuse.vp = c->vp; fuse.inv_alpha = c->inv_alpha_s; fuse.vq = c->vq;
    fuse.part = c->partials + 2 * (size_t)c->part_cap;
    const bool split = c->n_blocks / ws.n_groups < 5;
    const size_t smem = tmu32_smem(s_chunk);
#define TKHP_TMU32(F, SP) k_atom_tmu32<F, SP><<<ws.n_groups, GT, smem, s>>>(ws, ws.gpos32, ws.stage_pos32, c->mu32, K, c->acc, \
                                                                          c->n_pad, s_chunk, c->sm_count, c->st, c->spec_iter, fuse)
    if (c->far_on) { if (split) TKHP_TMU32(true, true); else TKHP_TMU32(true, false); }
    else { if (split) TKHP_TMU32(false, true); else TKHP_TMU32(false, false); }
#undef TKHP_TMU32
    c->n_launches += 1;
    TKHP_CUDA(c, cudaGetLastError());
    return TKHP_OK;
}

// dynamic shared memory opt-in of every ATOM-mode pair kernel, once per context (the attribute is
// per device; tkhp_create calls this with the context's device current)
int atom_pairs_configure(Ctx *c) {
    const int big = 2 * ATOM_SMEM + 8192;
    TKHP_CUDA(c, cudaFuncSetAttribute(k_atom_pairs<float, MODE_FIELD>, cudaFuncAttributeMaxDynamicSharedMemorySize, big));
    TKHP_CUDA(c, cudaFuncSetAttribute(k_atom_pairs<double, MODE_TMU>, cudaFuncAttributeMaxDynamicSharedMemorySize, big));
    TKHP_CUDA(c, cudaFuncSetAttribute(k_atom_pairs<double, MODE_FIELD>, cudaFuncAttributeMaxDynamicSharedMemorySize, big));
    const int tmu = (int)tmu32_smem(atom_chunk_capacity(false, 0));
    TKHP_CUDA(c, cudaFuncSetAttribute(k_atom_tmu32<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, tmu));
    TKHP_CUDA(c, cudaFuncSetAttribute(k_atom_tmu32<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, tmu));
    TKHP_CUDA(c, cudaFuncSetAttribute(k_atom_tmu32<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, tmu));
    TKHP_CUDA(c, cudaFuncSetAttribute(k_atom_tmu32<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, tmu));
    return TKHP_OK;
}

int atom_tmatvec(Ctx *c, cudaStream_t s) {
    ClusterWs ws = get_ws(c);
    if (c->stored_t && c->p.precision != TKHP_FP64) return atom_stored_tmatvec(c, s);      // TKHP_SOLVER_STORED_T
    return c->p.precision != TKHP_FP64 ? launch_tmu32(c, ws, s) : launch_atom_pairs<double, MODE_TMU>(c, ws, s);
}

int atom_field(Ctx *c, cudaStream_t s) {
    ClusterWs ws = get_ws(c);
    return c->p.precision != TKHP_FP64 ? launch_atom_pairs<float, MODE_FIELD>(c, ws, s)
                                        : launch_atom_pairs<double, MODE_FIELD>(c, ws, s);
}

}  // namespace tkhp
