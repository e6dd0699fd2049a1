// atom_pairs.cu -- ATOM list mode: exact per-atom lists and the pair kernels that walk them.
//
// Paper, "List filtering": a group's neighbour list is filtered down to "a list of
// atoms which really belong to a group's neighborhood", padded with phantom atoms, at the price of
// "a loss of coalesced memory access pattern".  CLUSTER mode (cluster.cuh) filters per 8-atom
// cluster, which still leaves ~52 % of the evaluated (atom, list atom) slots outside r_c.  ATOM
// mode carries the filtering to the end:
//  * the list is per ATOM and exact: every entry is a pair with R^2 <= r_c^2 for the positions of
//    the build (a list is only ever used for those positions), so the pair kernels contain no
//    cutoff test, no predicate and no select -- padding entries point at a dummy record with
//    zero payload;
//  * a CTA owns a group of <= 8 consecutive 32-atom blocks (one warp each) and stages the group's
//    neighbourhood ONCE in shared memory, already shifted into the group's frame (no image
//    arithmetic in the loop).  A lane owns one atom and only ever updates that atom: no atomics,
//    bit-reproducible results;
//  * entries are 16-bit BYTE OFFSETS into the staged chunk, stored per block as
//    [entry/4][lane][entry%4]: one coalesced 8-byte load per lane fetches 4 entries, fetched one
//    step ahead of their use;
//  * the loss of coalescing the paper notes becomes per-lane LDS.128 gathers from shared memory;
//    two pairs are evaluated together per lane (two independent dependency chains);
//  * FP32 partial sums are flushed into FP64 registers every 32 entries.
// The lists are built from the CLUSTER lists (the 8-atom-cluster list is the candidate set of
// each of its atoms): k_atom_lists below.
#include "cluster.cuh"
#include "reduce.cuh"

namespace tkhp {

constexpr int MODE_TMU = 0, MODE_FIELD = 1;
static_assert(GT == RED_THREADS, "the fused PCG epilogue uses the 256-thread block reductions");

// PCG fusion (MODE_TMU): the lane that owns atom i holds (T p)_i when the
// list is exhausted, so q_i = p_i/alpha_i - (T p)_i - self p_i and the block's share of p.q are
// formed here instead of in a separate vector kernel.
struct PcgFuse {
    int on;
    double self;
    const double *vp;          // 3 n_pad, direction p (FP64)
    const double *inv_alpha;   // n_pad
    double *vq;                // 3 n_pad out
    double *part;              // 2 * n_groups block partials
};

// ----------------------------------------------------------------------------- list construction
// One CTA per group.  Chunk by chunk, the staged positions are put in shared memory, every lane
// walks its cluster's list (staging order) and appends the byte offset of each atom within r_c of
// ITS atom to its own list; the warp then pads all 32 lists of the chunk to a common length
// (multiple of 4).  The test is the pair kernels' own arithmetic (group-frame coordinates, FP32 in
// MIXED, FP64 in FP64 mode).
template <typename real>
__global__ void __launch_bounds__(GT)
k_atom_lists(ClusterWs ws, const typename Vec4<real>::type *__restrict__ gpos,
             const typename Vec4<real>::type *__restrict__ stage_pos, real rc2, DeviceState *st) {
    using vec4 = typename Vec4<real>::type;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    vec4 *s_pos = reinterpret_cast<vec4 *>(smem_raw);

    const int g = blockIdx.x, t = threadIdx.x, lane = t & 31, w = t >> 5;
    const int b0 = ws.group_first[g], nb = ws.group_first[g + 1] - b0;
    const int count = ws.stage_count[g];
    const size_t gbase = (size_t)g * ws.s_cap;
    const int s_chunk = atom_chunk_capacity(sizeof(real) == 8, ws.chunk_cap);
    const int n_chunks = atom_chunks_of(count, s_chunk);
    if (n_chunks > NCH_MAX) {                      // uniform over the CTA
        if (t == 0) st->atom_bad = 1;
        return;
    }
    const unsigned magic = ((1u << 20) + (unsigned)n_chunks - 1u) / (unsigned)n_chunks;   // e / n for e < 2^16
    const bool active = w < nb;
    const int blk = b0 + (active ? w : 0);
    const int slot = blk * BLOCK + lane;
    const vec4 pi = gpos[slot];
    const int oct = slot >> 3;
    const int L = active ? ws.oct_len[oct] : 0;
    const uint16_t *__restrict__ ent = ws.entries + (size_t)oct * ws.l_cap;
    // a lane's list as quads of 4 entries: quad q of lane l at uint2 index q * 32 + l of the block
    uint2 *__restrict__ out = reinterpret_cast<uint2 *>(ws.alist + (size_t)blk * ws.a_cap * 32) + lane;
    int32_t *__restrict__ arow = ws.arow + (size_t)blk * (NCH_MAX + 1);
    const unsigned dummy = (unsigned)s_chunk * (unsigned)sizeof(vec4);
    const unsigned long long dummy4 = 0x0001000100010001ull * (unsigned long long)dummy;
    const int q_cap = ws.a_cap >> 2;
    const uint4 *__restrict__ ent8 = reinterpret_cast<const uint4 *>(ent);    // 8 entries per load
    const int L8 = L >> 3;                                                     // L is a multiple of 8

    int q0 = 0;        // first quad of the current chunk's list (same for all lanes)
    for (int c = 0; c < n_chunks; ++c) {
        __syncthreads();
        for (int l = t, idx = c + t * n_chunks; idx < count; l += GT, idx += GT * n_chunks)
            s_pos[l] = stage_pos[gbase + idx];
        __syncthreads();
        if (!active) continue;
        if (lane == 0) arow[c] = q0 << 2;
        int k = 0;                         // entries this lane appended in this chunk
        unsigned long long pend = 0;       // the quad being filled
        uint4 nxt = L8 > 0 ? ent8[0] : make_uint4(0, 0, 0, 0);
        bool open = true;
        for (int v = 0; v < L8 && open; ++v) {
            const uint4 cur = nxt;
            if (v + 1 < L8) nxt = ent8[v + 1];           // one address per quarter warp, one load ahead
            const unsigned word[4] = {cur.x, cur.y, cur.z, cur.w};
#pragma unroll
            for (int h = 0; h < 8; ++h) {
                const unsigned e = (word[h >> 1] >> ((h & 1) * 16)) & 0xffffu;
                if ((int)e >= count) { open = false; break; }      // padding entries (== count) close the list
                const unsigned loc = (e * magic) >> 20;            // e / n_chunks
                if (e - loc * (unsigned)n_chunks != (unsigned)c) continue;
                const vec4 pj = s_pos[loc];
                const real Rx = pi.x - pj.x, Ry = pi.y - pj.y, Rz = pi.z - pj.z;
                const real r2 = Rx * Rx + Ry * Ry + Rz * Rz;
                if (r2 <= rc2 && r2 > (real)1e-10) {
                    pend |= (unsigned long long)(loc * (unsigned)sizeof(vec4)) << ((k & 3) * 16);
                    if ((k & 3) == 3) {
                        const int q = q0 + (k >> 2);
                        if (q < q_cap) out[(size_t)q * 32] = make_uint2((unsigned)pend, (unsigned)(pend >> 32));
                        pend = 0;
                    }
                    ++k;
                }
            }
        }
        int kmax = k;
        for (int o = 16; o > 0; o >>= 1) kmax = max(kmax, __shfl_xor_sync(0xffffffffu, kmax, o));
        int qmax = ((kmax + 7) >> 3) << 1;      // even: the pair kernels take two quads per trip
        if (q0 + qmax > q_cap) {
            if (lane == 0) st->atom_bad = 1;
            qmax = q_cap - q0;
        }
        int qd = k >> 2;                   // first quad this lane has not stored yet
        if ((k & 3) != 0) {                // partly filled quad: the rest are dummies
            pend |= dummy4 << ((k & 3) * 16);
            if (q0 + qd < q_cap) out[(size_t)(q0 + qd) * 32] = make_uint2((unsigned)pend, (unsigned)(pend >> 32));
            ++qd;
        }
        for (; qd < qmax; ++qd) out[(size_t)(q0 + qd) * 32] = make_uint2((unsigned)dummy4, (unsigned)(dummy4 >> 32));
        q0 += qmax;
    }
    const int k0 = q0 << 2;
    if (active && lane == 0) {
        for (int c = n_chunks; c <= NCH_MAX; ++c) arow[c] = k0;
        atomicAdd((unsigned long long *)&st->n_atom_entries, (unsigned long long)k0);
    }
}

// ----------------------------------------------------------------------------- bank-aware order
// The pair kernels gather 16-byte records from shared memory, one per lane and step.  A quarter
// warp (8 lanes) is served in one wavefront only if its 8 records fall into 8 different bank
// groups (record index mod 8); with the lists in staging order they are random and an LDS.128
// costs 2.35 wavefronts instead of 1 (ncu, r01).  k_atom_reorder permutes every lane's list, per
// chunk and in place, so that at step t lane l reads a record of bank group (t + l) mod 8 whenever
// it has one left: entries are dealt into 8 per-bank columns of rows t = ((b - l) mod 8) + 8 r;
// entries of over-full columns (rows beyond the common padded length) move into the holes of
// under-full ones (those steps may conflict), the remaining holes are the padding.  The set of
// entries of a list does not change, only their order, so the result changes by FP32 summation
// order only.  One warp per 32-atom block, list columns in shared memory ([row][lane], u16).
constexpr int RO_ROWS = 256;          // rows per lane the shared-memory image can hold
constexpr int RO_WARPS = 4;

__global__ void __launch_bounds__(RO_WARPS * 32)
k_atom_reorder(ClusterWs ws, int n_blocks, int rec_bytes, int s_chunk) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int blk = blockIdx.x * RO_WARPS + w;
    if (blk >= n_blocks) return;
    uint16_t *img = reinterpret_cast<uint16_t *>(smem_raw) + (size_t)w * RO_ROWS * 32 + lane;   // img[row * 32]
    uint2 *__restrict__ list = reinterpret_cast<uint2 *>(ws.alist + (size_t)blk * ws.a_cap * 32) + lane;
    const int32_t *__restrict__ arow = ws.arow + (size_t)blk * (NCH_MAX + 1);
    const unsigned dummy = (unsigned)s_chunk * (unsigned)rec_bytes;
    const int l8 = lane & 7;

    for (int c = 0; c < NCH_MAX; ++c) {
        const int q0 = arow[c] >> 2, q1 = arow[c + 1] >> 2;
        const int len = (q1 - q0) << 2;                    // common padded length of this chunk's lists
        if (len <= 0) continue;
        if (len > RO_ROWS) continue;                       // image too small: keep staging order
        for (int r = 0; r < RO_ROWS; ++r) img[r * 32] = 0xffffu;
        // deal the entries into the per-bank columns
        unsigned long long cnt = 0;                        // 8 counters of 8 bits
        bool fits = true;
        for (int q = q0; q < q1; ++q) {
            const uint2 e = list[(size_t)q * 32];
            const unsigned v[4] = {e.x & 0xffffu, e.x >> 16, e.y & 0xffffu, e.y >> 16};
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                if (v[h] == dummy) continue;
                const unsigned b = (v[h] >> 4) & 7u;
                const unsigned r = (unsigned)(cnt >> (8 * b)) & 0xffu;
                const unsigned t = ((b - (unsigned)l8) & 7u) + 8u * r;
                if (t < (unsigned)RO_ROWS) img[t * 32] = (uint16_t)v[h]; else fits = false;
                cnt += 1ull << (8 * b);
            }
        }
        if (!__all_sync(0xffffffffu, fits)) continue;      // (never seen) a column ran past the image
        // over-full columns -> holes of under-full ones
        const unsigned R = (unsigned)len >> 3;             // rows each column keeps
        unsigned hb = 0, hr = (unsigned)cnt & 0xffu;       // hole cursor: column hb, row hr
        for (unsigned b = 0; b < 8; ++b) {
            const unsigned cb = (unsigned)(cnt >> (8 * b)) & 0xffu;
            for (unsigned r = R; r < cb; ++r) {
                const unsigned t = ((b - (unsigned)l8) & 7u) + 8u * r;
                const uint16_t v = img[t * 32];
                while (hr >= R) { ++hb; hr = (unsigned)(cnt >> (8 * hb)) & 0xffu; }
                img[(((hb - (unsigned)l8) & 7u) + 8u * hr) * 32] = v;
                ++hr;
            }
        }
        // write back; untouched holes (0xffff) are the padding
        for (int q = q0; q < q1; ++q) {
            unsigned v[4];
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                const unsigned x = img[(((q - q0) << 2) + h) * 32];
                v[h] = x == 0xffffu ? dummy : x;
            }
            list[(size_t)q * 32] = make_uint2(v[0] | (v[1] << 16), v[2] | (v[3] << 16));
        }
        __syncwarp();
    }
}

// ----------------------------------------------------------------------------- pair kernels
//   MODE_TMU   (T1,T2): out_i += -m1 mu_j + m2 (mu_j.R) R            staged: pos+w, mu
//   MODE_FIELD (F1,F2): field at i from (q,d,Q)_j, same-group pairs contribute zero here (the FP64
//                       correction pass adds them, pcg.cu)            staged: pos+w, 3 multipole vec4
template <typename real, int MODE, int W>
__device__ __forceinline__ void eval_pairs(const unsigned char *s_base, int pay_stride, const unsigned (&off)[W],
                                           const typename Vec4<real>::type &pi, real gi,
                                           const PairConsts<real> &kc, real &ax, real &ay, real &az) {
    using vec4 = typename Vec4<real>::type;
    constexpr int NK = MODE == MODE_TMU ? 2 : 3;
    vec4 pj[W];
    real Rx[W], Ry[W], Rz[W], r2[W], ww[W], G[W][NK];
#pragma unroll
    for (int u = 0; u < W; ++u) pj[u] = *reinterpret_cast<const vec4 *>(s_base + off[u]);
    if (MODE == MODE_TMU) {
        vec4 mj[W];
#pragma unroll
        for (int u = 0; u < W; ++u) mj[u] = *reinterpret_cast<const vec4 *>(s_base + pay_stride + off[u]);
#pragma unroll
        for (int u = 0; u < W; ++u) {
            Rx[u] = pi.x - pj[u].x; Ry[u] = pi.y - pj[u].y; Rz[u] = pi.z - pj[u].z;
            r2[u] = Rx[u] * Rx[u] + Ry[u] * Ry[u] + Rz[u] * Rz[u];
            ww[u] = pi.w * pj[u].w;
        }
        radial_w<NK, W>(r2, ww, kc, G);
#pragma unroll
        for (int u = 0; u < W; ++u)
            tmu_apply<real>(G[u][0], G[u][1], Rx[u], Ry[u], Rz[u], mj[u].x, mj[u].y, mj[u].z, ax, ay, az);
    } else {
        vec4 b0v[W], b1v[W], b2v[W];
        bool in[W];
#pragma unroll
        for (int u = 0; u < W; ++u) {
            b0v[u] = *reinterpret_cast<const vec4 *>(s_base + pay_stride + off[u]);
            b1v[u] = *reinterpret_cast<const vec4 *>(s_base + 2 * pay_stride + off[u]);
            b2v[u] = *reinterpret_cast<const vec4 *>(s_base + 3 * pay_stride + off[u]);
        }
#pragma unroll
        for (int u = 0; u < W; ++u) {
            Rx[u] = pi.x - pj[u].x; Ry[u] = pi.y - pj[u].y; Rz[u] = pi.z - pj[u].z;
            r2[u] = Rx[u] * Rx[u] + Ry[u] * Ry[u] + Rz[u] * Rz[u];
            ww[u] = pi.w * pj[u].w;
            in[u] = b2v[u].z != gi;
        }
        radial_w<NK, W>(r2, ww, kc, G);
#pragma unroll
        for (int u = 0; u < W; ++u) {
            if (!in[u]) { G[u][0] = 0; G[u][1] = 0; G[u][2] = 0; }
            field_apply<real>(G[u], Rx[u], Ry[u], Rz[u], b0v[u].x, b0v[u].y, b0v[u].z, b0v[u].w, b1v[u].x,
                              b1v[u].y, b1v[u].z, b1v[u].w, b2v[u].x, b2v[u].y, ax, ay, az);
        }
    }
}

// pairs evaluated together per lane (independent dependency chains): 4 in the FP32 T.mu kernel
// (a 98k-atom system has only ~21 warps per SM, so the latency must be covered inside the warp),
// 2 elsewhere (register budget)
template <typename real, int MODE> struct PairWidth { static constexpr int W = 2; };
template <> struct PairWidth<float, MODE_TMU> { static constexpr int W = 2; };   // 4 measured slower (80 registers)

// one lane's quad of list entries (8 bytes), read-only path, pinned in program order
__device__ __forceinline__ uint2 ldg_list(const uint2 *p) {
    uint2 v;
    asm volatile("ld.global.nc.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p));
    return v;
}

template <typename real, int MODE>
__device__ __forceinline__ void eval_quad(const unsigned char *s_base, int pay_stride, uint2 e,
                                          const typename Vec4<real>::type &pi, real gi,
                                          const PairConsts<real> &kc, real &ax, real &ay, real &az) {
    if (PairWidth<real, MODE>::W == 4) {
        const unsigned off[4] = {e.x & 0xffffu, e.x >> 16, e.y & 0xffffu, e.y >> 16};
        eval_pairs<real, MODE, 4>(s_base, pay_stride, off, pi, gi, kc, ax, ay, az);
    } else {
        const unsigned o0[2] = {e.x & 0xffffu, e.x >> 16}, o1[2] = {e.y & 0xffffu, e.y >> 16};
        eval_pairs<real, MODE, 2>(s_base, pay_stride, o0, pi, gi, kc, ax, ay, az);
        eval_pairs<real, MODE, 2>(s_base, pay_stride, o1, pi, gi, kc, ax, ay, az);
    }
}

// resident CTAs per SM the register allocation must allow: FP32 T.mu 4 (<= 64 registers; shared
// memory allows 4 x 56 KB), FP32 field 2 (112 KB of staging), FP64 1
template <typename real, int MODE> struct MinCtas { static constexpr int N = sizeof(real) == 8 ? 1 : (MODE == MODE_TMU ? 3 : 2); };

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
    constexpr int SU = 2;         // staging loads in flight per thread
    extern __shared__ __align__(16) unsigned char smem_raw[];
    vec4 *s_pos = reinterpret_cast<vec4 *>(smem_raw);          // [s_chunk + 1], last = dummy
    vec4 *s_pay = s_pos + (s_chunk + 1);                       // NPAY arrays of [s_chunk + 1]
    const int pstride = s_chunk + 1;
    const int pay_stride = pstride * (int)sizeof(vec4);

    const int g = blockIdx.x, t = threadIdx.x, lane = t & 31, w = t >> 5;
    const int b0 = ws.group_first[g], nb = ws.group_first[g + 1] - b0;
    const int count = ws.stage_count[g];
    const int n_chunks = atom_chunks_of(count, s_chunk);
    const size_t gbase = (size_t)g * ws.s_cap;
    const bool active = w < nb;
    const int blk = b0 + (active ? w : 0);
    const int slot = blk * BLOCK + lane;
    const vec4 pi = gpos[slot];
    real gi = 0;
    if (MODE == MODE_FIELD) gi = data[2 * (size_t)n_pad + slot].z;
    const uint2 *__restrict__ lp = reinterpret_cast<const uint2 *>(ws.alist + (size_t)blk * ws.a_cap * 32) + lane;
    const int32_t *__restrict__ arow = ws.arow + (size_t)blk * (NCH_MAX + 1);

    double dx = 0.0, dy = 0.0, dz = 0.0;
    real ax = 0, ay = 0, az = 0;
    int since_flush = 0;

    if (t == 0) {                              // permanent dummy record: far away, zero payload
        vec4 far, zero;
        far.x = far.y = far.z = (real)(-2.0f * PHANTOM_FAR); far.w = 0;
        zero.x = zero.y = zero.z = zero.w = 0;
        s_pos[s_chunk] = far;
        for (int k = 0; k < NPAY; ++k) s_pay[k * pstride + s_chunk] = zero;
    }

    for (int c = 0; c < n_chunks; ++c) {
        __syncthreads();
        // gather of the payload by staged atom: SU records per thread in flight (index, then payload)
        for (int l0 = t, i0 = c + t * n_chunks; i0 < count; l0 += SU * GT, i0 += SU * GT * n_chunks) {
            int a[SU];
            vec4 p[SU];
#pragma unroll
            for (int u = 0; u < SU; ++u) {
                const int idx = i0 + u * GT * n_chunks;
                const bool ok = idx < count;
                a[u] = ok ? ws.stage_atom[gbase + idx] : -1;
                if (ok) p[u] = stage_pos[gbase + idx];
            }
#pragma unroll
            for (int k = 0; k < NPAY; ++k) {
                vec4 d[SU];
#pragma unroll
                for (int u = 0; u < SU; ++u)
                    if (a[u] >= 0) d[u] = data[(size_t)k * n_pad + a[u]];
#pragma unroll
                for (int u = 0; u < SU; ++u)
                    if (a[u] >= 0) s_pay[k * pstride + l0 + u * GT] = d[u];
            }
#pragma unroll
            for (int u = 0; u < SU; ++u)
                if (a[u] >= 0) s_pos[l0 + u * GT] = p[u];
        }
        __syncthreads();
        if (!active) continue;
        const int q0 = arow[c] >> 2, q1 = arow[c + 1] >> 2;
        if (q0 >= q1) continue;
        const unsigned char *s_base = smem_raw;
        // Two quads per trip; a quad is loaded one whole trip (8 pairs) before its use, right after
        // the registers it goes to have been unpacked.  The loads are
        // volatile asm so that they stay where they are written: a load that drifts to the end of
        // the loop body shares its scoreboard with the unpack at the top and exposes the full L2
        // latency in every trip (measured: 30 % of all stall samples).
        const uint2 *pq = lp + (size_t)q0 * 32;
        const uint2 *const pend = lp + (size_t)(q1 - 1) * 32;      // clamp for the look-ahead loads
        uint2 eA = ldg_list(pq);
        uint2 eB = ldg_list(pq + 32);
        for (int q = q0; q < q1; q += 2, pq += 64) {
            const uint2 a = eA;
            eA = ldg_list(pq + 64 <= pend ? pq + 64 : pend);
            eval_quad<real, MODE>(s_base, pay_stride, a, pi, gi, kc, ax, ay, az);
            const uint2 b = eB;
            eB = ldg_list(pq + 96 <= pend ? pq + 96 : pend);
            eval_quad<real, MODE>(s_base, pay_stride, b, pi, gi, kc, ax, ay, az);
            if (++since_flush == 4) {          // every 32 entries: FP32 partial -> FP64 accumulator
                dx += (double)ax; dy += (double)ay; dz += (double)az;
                ax = 0; ay = 0; az = 0;
                since_flush = 0;
            }
        }
    }
    dx += (double)ax; dy += (double)ay; dz += (double)az;
    if (active) {
        acc[slot] = dx;
        acc[n_pad + slot] = dy;
        acc[2 * (size_t)n_pad + slot] = dz;
    }
    if (MODE == MODE_TMU && fuse.on) {
        double pq = 0, dummy = 0;
        if (active) {
            const double ia = fuse.inv_alpha[slot];
            const double d[3] = {dx, dy, dz};
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const size_t o = (size_t)k * n_pad + slot;
                const double p = fuse.vp[o];
                const double q = p * ia - d[k] - fuse.self * p;
                fuse.vq[o] = q;
                pq += p * q;
            }
        }
        block_sum2(pq, dummy);
        if (grid_sum2_last_block(fuse.part, &st->ticket, pq, dummy) && threadIdx.x == 0) st->pq = pq;
    }
}

// ----------------------------------------------------------------------------- host side
int atom_build(Ctx *c, cudaStream_t s) {
    ClusterWs ws = get_ws(c);
    const bool f64 = c->p.precision == TKHP_FP64;
    const int s_chunk = atom_chunk_capacity(f64, ws.chunk_cap);
    const size_t smem = (size_t)s_chunk * (f64 ? sizeof(double4) : sizeof(float4));
    const double rc2 = c->p.cutoff * c->p.cutoff;
    if (f64)
        k_atom_lists<double><<<ws.n_groups, GT, smem, s>>>(ws, ws.gpos64, ws.stage_pos64, rc2, c->st);
    else
        k_atom_lists<float><<<ws.n_groups, GT, smem, s>>>(ws, ws.gpos32, ws.stage_pos32, (float)rc2, c->st);
    static bool ro_configured = false;
    const size_t ro_smem = (size_t)RO_WARPS * RO_ROWS * 32 * sizeof(uint16_t);
    if (!ro_configured) {
        TKHP_CUDA(c, cudaFuncSetAttribute(k_atom_reorder, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ro_smem));
        ro_configured = true;
    }
    k_atom_reorder<<<div_up(c->n_blocks, RO_WARPS), RO_WARPS * 32, ro_smem, s>>>(ws, c->n_blocks, f64 ? 32 : 16, s_chunk);
    c->n_launches += 2;
    TKHP_CUDA(c, cudaGetLastError());
    return TKHP_OK;
}

template <typename real, int MODE>
static int launch_atom_pairs(Ctx *c, const ClusterWs &ws, cudaStream_t s) {
    using vec4 = typename Vec4<real>::type;
    constexpr int NPAY = MODE == MODE_TMU ? 1 : 3;
    constexpr int which = sizeof(real) == 8;
    const int s_chunk = atom_chunk_capacity(which, ws.chunk_cap);
    const size_t smem = sizeof(vec4) * (size_t)(1 + NPAY) * (size_t)(s_chunk + 1);
    static bool configured[2][2] = {{false, false}, {false, false}};
    if (!configured[which][MODE]) {
        TKHP_CUDA(c, cudaFuncSetAttribute(k_atom_pairs<real, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          2 * ATOM_SMEM + 4096));
        configured[which][MODE] = true;
    }
    PairConsts<real> k;
    k.beta = (real)c->p.ewald_beta;
    k.c1 = (real)(2.0 / SQRT_PI);
    k.c23 = (real)(4.0 / (3.0 * SQRT_PI));
    k.rc2 = (real)(c->p.cutoff * c->p.cutoff);
    k.box = (real)1;
    k.inv_box = (real)0;
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

int atom_tmatvec(Ctx *c, cudaStream_t s) {
    ClusterWs ws = get_ws(c);
    return c->p.precision == TKHP_MIXED ? launch_atom_pairs<float, MODE_TMU>(c, ws, s)
                                        : launch_atom_pairs<double, MODE_TMU>(c, ws, s);
}

int atom_field(Ctx *c, cudaStream_t s) {
    ClusterWs ws = get_ws(c);
    return c->p.precision == TKHP_MIXED ? launch_atom_pairs<float, MODE_FIELD>(c, ws, s)
                                        : launch_atom_pairs<double, MODE_FIELD>(c, ws, s);
}

long long atom_slots(Ctx *c) { return 32LL * c->h_state->n_atom_entries; }

}  // namespace tkhp
