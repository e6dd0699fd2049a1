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
//    [entry/8][lane][entry%8]: 16 bytes per lane and trip of 8 pairs, a coalesced 512-byte row per
//    warp.  The FP32 T.mu kernel streams the rows through a per-warp shared-memory ring with
//    cp.async, several trips ahead (the L2/HBM latency of this stream was the largest stall of
//    the register-prefetch version); the other variants load them one trip ahead into registers;
//  * the loss of coalescing the paper notes becomes per-lane LDS.128 gathers from shared memory;
//    two pairs are evaluated together per lane: in the FP32 T.mu kernel as the two halves of
//    packed FP32 instructions (f32x2.cuh), elsewhere as two independent dependency chains;
//  * a group with fewer than 5 blocks gives every block to 2, 4 or 8 warps (interleaved list rows);
//  * FP32 partial sums are flushed into FP64 registers every 32 entries.
// The lists are built from the CLUSTER lists (the 8-atom-cluster list is the candidate set of
// each of its atoms): k_atom_lists below.
#include "cluster.cuh"
#include "f32x2.cuh"
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
// quad q (4 entries) of a lane, as uint2 index relative to the lane's first quad (lane * 2)
__host__ __device__ __forceinline__ size_t qidx(int q) { return (size_t)(q >> 1) * 64 + (size_t)(q & 1); }

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
    // a lane's list as quads of 4 entries: quad q of lane l at uint2 index qidx(q) + 2 l of the block
    uint2 *__restrict__ out = reinterpret_cast<uint2 *>(ws.alist + (size_t)blk * ws.a_cap * 32) + lane * 2;
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
            // the 8 entries of the vector are tested together (8 independent chains: the loop was bound
            // by fixed-latency dependencies), then the hits are appended in list order
            unsigned loc[8];
            bool hit[8];
#pragma unroll
            for (int h = 0; h < 8; ++h) {
                const unsigned e = (word[h >> 1] >> ((h & 1) * 16)) & 0xffffu;
                loc[h] = (e * magic) >> 20;                        // e / n_chunks
                hit[h] = (int)e < count && e - loc[h] * (unsigned)n_chunks == (unsigned)c;   // padding entries are == count
                if (h == 7) open = (int)e < count;                 // padding only at the end of a list
            }
#pragma unroll
            for (int h = 0; h < 8; ++h) {
                const vec4 pj = s_pos[hit[h] ? loc[h] : 0u];
                const real Rx = pi.x - pj.x, Ry = pi.y - pj.y, Rz = pi.z - pj.z;
                const real r2 = Rx * Rx + Ry * Ry + Rz * Rz;
                hit[h] = hit[h] && r2 <= rc2 && r2 > (real)1e-10;
            }
#pragma unroll
            for (int h = 0; h < 8; ++h) {
                if (hit[h]) {
                    pend |= (unsigned long long)(loc[h] * (unsigned)sizeof(vec4)) << ((k & 3) * 16);
                    if ((k & 3) == 3) {
                        const int q = q0 + (k >> 2);
                        if (q < q_cap) out[qidx(q)] = make_uint2((unsigned)pend, (unsigned)(pend >> 32));
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
            if (q0 + qd < q_cap) out[qidx(q0 + qd)] = make_uint2((unsigned)pend, (unsigned)(pend >> 32));
            ++qd;
        }
        for (; qd < qmax; ++qd) out[qidx(q0 + qd)] = make_uint2((unsigned)dummy4, (unsigned)(dummy4 >> 32));
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
    uint2 *__restrict__ list = reinterpret_cast<uint2 *>(ws.alist + (size_t)blk * ws.a_cap * 32) + lane * 2;
    const int32_t *__restrict__ arow = ws.arow + (size_t)blk * (NCH_MAX + 1);
    const unsigned dummy = (unsigned)s_chunk * (unsigned)rec_bytes;
    const int l8 = lane & 7;

    for (int c = 0; c < NCH_MAX; ++c) {
        const int q0 = arow[c] >> 2, q1 = arow[c + 1] >> 2;
        const int len = (q1 - q0) << 2;                    // common padded length of this chunk's lists
        if (len <= 0) continue;
        if (len > RO_ROWS) continue;                       // image too small: keep staging order
        for (int r = 0; r < len; ++r) img[r * 32] = 0xffffu;     // rows >= len are only read where written
        // deal the entries into the per-bank columns; a list row (8 entries = 16 B per lane) is
        // loaded one row ahead of its use
        unsigned long long cnt = 0;                        // 8 counters of 8 bits
        bool fits = true;
        const uint4 *rowp = reinterpret_cast<const uint4 *>(list + qidx(q0));      // q0 is even: row q0 / 2
        uint4 nxt = rowp[0];
        for (int q = q0; q < q1; q += 2, rowp += 32) {
            const uint4 e = nxt;
            if (q + 2 < q1) nxt = rowp[32];
            const unsigned v[8] = {e.x & 0xffffu, e.x >> 16, e.y & 0xffffu, e.y >> 16,
                                   e.z & 0xffffu, e.z >> 16, e.w & 0xffffu, e.w >> 16};
#pragma unroll
            for (int h = 0; h < 8; ++h) {
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
        uint4 *outp = reinterpret_cast<uint4 *>(list + qidx(q0));
        for (int q = q0; q < q1; q += 2, outp += 32) {
            unsigned v[8];
#pragma unroll
            for (int h = 0; h < 8; ++h) {
                const unsigned x = img[(((q - q0) << 2) + h) * 32];
                v[h] = x == 0xffffu ? dummy : x;
            }
            *outp = make_uint4(v[0] | (v[1] << 16), v[2] | (v[3] << 16), v[4] | (v[5] << 16), v[6] | (v[7] << 16));
        }
        __syncwarp();
    }
}

// ----------------------------------------------------------------------------- pair kernels
//   MODE_TMU   (T1,T2): out_i += -m1 mu_j + m2 (mu_j.R) R            staged: pos+w, mu
//   MODE_FIELD (F1,F2): field at i from (q,d,Q)_j, same-group pairs contribute zero here (the FP64
//                       correction pass adds them, pcg.cu)            staged: pos+w, 3 multipole vec4
// ---- FP32 partial sums of one lane ------------------------------------------------------------
// Generic: one (x, y, z) partial.  Packed FP32 T.mu: two partials, C = sum G2/3 (mu_j.D) D and
// M = sum G1 mu_j (D = r_j - r_i), so that the pair loop needs neither the factor 3 nor a
// negation; (T mu)_i = 3 C - M is formed at every flush into the FP64 registers.
template <typename real, int MODE>
struct Partial {
    real x = 0, y = 0, z = 0;
    __device__ __forceinline__ void flush(double &dx, double &dy, double &dz) {
        dx += (double)x; dy += (double)y; dz += (double)z;
        x = 0; y = 0; z = 0;
    }
};
template <>
struct Partial<float, MODE_TMU> {
    f2 cxy = 0ull, mxy = 0ull;
    float cz = 0.f, mz = 0.f;
    __device__ __forceinline__ void flush(double &dx, double &dy, double &dz) {
        dx += (double)fmaf(3.0f, lo(cxy), -lo(mxy));
        dy += (double)fmaf(3.0f, hi(cxy), -hi(mxy));
        dz += (double)fmaf(3.0f, cz, -mz);
        cxy = 0ull; mxy = 0ull; cz = 0.f; mz = 0.f;
    }
};

// ---- packed FP32 T.mu: two list entries of one lane per call ------------------------------------
// The two pairs (j0, j1) of a lane share every instruction of the radial chain (lo half = j0,
// hi half = j1); the geometry and the 3-vector updates are packed over (x, y), the pair LDS.128
// delivers them in.  Per pair: 25 FMA-pipe issue slots (41 pipe cycles) + 4 MUFU, against 46
// scalar instructions.  Per-lane constants: pxy = (x_i, y_i), nz0 = (-z_i, 0),
// one_w = (1, w_i log2 e) so that one FFMA2 gives (z_j - z_i, w_i w_j log2 e).
struct TmuLane {
    f2 pxy, nz0, one_w;
};
struct TmuConsts {
    float pb;       // P beta (TKHP_ERFCX_P): u = 1 / (1 + pb R)
    float nb2l;     // -beta^2 log2 e:        e^{-z^2} = ex2(nb2l R^2)
    float c1b;      // (2/sqrt pi) beta:      c z
    float k3;       // (4/(3 sqrt pi)) beta^3: (2c/3) z^3 = k3 R^3
};

__device__ __forceinline__ void tmu_pair2(const unsigned char *s_base, int pay_stride, unsigned off0, unsigned off1,
                                          const TmuLane &L, const TmuConsts &K, Partial<float, MODE_TMU> &A) {
    constexpr float c[TKHP_ERFCX_DEG + 1] = TKHP_ERFCX_COEFFS;
    constexpr float LN2 = 0.69314718055994531f;
    const ulonglong2 p0 = *reinterpret_cast<const ulonglong2 *>(s_base + off0);               // (x,y) (z,w)
    const ulonglong2 p1 = *reinterpret_cast<const ulonglong2 *>(s_base + off1);
    const ulonglong2 m0 = *reinterpret_cast<const ulonglong2 *>(s_base + pay_stride + off0);  // (mx,my) (mz,0)
    const ulonglong2 m1 = *reinterpret_cast<const ulonglong2 *>(s_base + pay_stride + off1);
    const f2 Dxy0 = sub2(p0.x, L.pxy), Dxy1 = sub2(p1.x, L.pxy);
    const f2 Dzw0 = fma2(p0.y, L.one_w, L.nz0), Dzw1 = fma2(p1.y, L.one_w, L.nz0);
    float s0 = lo(Dxy0) * lo(Dxy0), s1 = lo(Dxy1) * lo(Dxy1);
    s0 = fmaf(hi(Dxy0), hi(Dxy0), s0); s1 = fmaf(hi(Dxy1), hi(Dxy1), s1);
    s0 = fmaf(lo(Dzw0), lo(Dzw0), s0); s1 = fmaf(lo(Dzw1), lo(Dzw1), s1);
    const f2 r2 = pk(s0, s1);
    const f2 rinv = pk(fast_rsqrt(s0), fast_rsqrt(s1));
    const f2 r = mul2(r2, rinv);
    const f2 ua = fma2(r, bc(K.pb), bc(1.0f));
    const f2 u = pk(fast_rcp(lo(ua)), fast_rcp(hi(ua)));
    const f2 ea = mul2(r2, bc(K.nb2l));
    const f2 ez = pk(fast_ex2(lo(ea)), fast_ex2(hi(ea)));
    const f2 r3 = mul2(r2, r);
    const f2 xl = pk(lo(r3) * hi(Dzw0), hi(r3) * hi(Dzw1));         // x log2 e
    const f2 et = pk(fast_ex2(-lo(xl)), fast_ex2(-hi(xl)));
    f2 p = bc(c[TKHP_ERFCX_DEG]);
#pragma unroll
    for (int d = TKHP_ERFCX_DEG - 1; d >= 0; --d) p = fma2(p, u, bc(c[d]));
    const f2 g1 = fma2(r, bc(K.c1b), p);                             // erfcx(z) + c z
    const f2 a1 = fma2(ez, g1, neg2(et));                            // R^3 G1
    const f2 h2 = fma2(r3, bc(K.k3), g1);
    const f2 x = mul2(xl, bc(LN2));
    const f2 xe = fma2(x, et, et);                                   // (1 + x) e^-x
    const f2 b2 = fma2(ez, h2, neg2(xe));                            // R^5 G2 / 3
    const f2 rinv2 = mul2(rinv, rinv);
    const f2 rinv3 = mul2(rinv2, rinv);
    const f2 G1 = mul2(a1, rinv3);
    const f2 G2 = mul2(b2, mul2(rinv2, rinv3));                      // G2 / 3
    float d0 = lo(m0.x) * lo(Dxy0), d1 = lo(m1.x) * lo(Dxy1);
    d0 = fmaf(hi(m0.x), hi(Dxy0), d0); d1 = fmaf(hi(m1.x), hi(Dxy1), d1);
    d0 = fmaf(lo(m0.y), lo(Dzw0), d0); d1 = fmaf(lo(m1.y), lo(Dzw1), d1);
    const f2 cc = mul2(G2, pk(d0, d1));
    A.cxy = fma2(Dxy0, bc(lo(cc)), A.cxy); A.cz = fmaf(lo(cc), lo(Dzw0), A.cz);
    A.mxy = fma2(m0.x, bc(lo(G1)), A.mxy); A.mz = fmaf(lo(G1), lo(m0.y), A.mz);
    A.cxy = fma2(Dxy1, bc(hi(cc)), A.cxy); A.cz = fmaf(hi(cc), lo(Dzw1), A.cz);
    A.mxy = fma2(m1.x, bc(hi(G1)), A.mxy); A.mz = fmaf(hi(G1), lo(m1.y), A.mz);
}

template <typename real, int MODE, int W>
__device__ __forceinline__ void eval_pairs(const unsigned char *s_base, int pay_stride, const unsigned (&off)[W],
                                           const typename Vec4<real>::type &pi, real gi,
                                           const PairConsts<real> &kc, Partial<real, MODE> &A) {
    using vec4 = typename Vec4<real>::type;
    constexpr int NK = MODE == MODE_TMU ? 2 : 3;
    real &ax = A.x, &ay = A.y, &az = A.z;
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

// one lane's quad of list entries (8 bytes), read-only path, pinned in program order
__device__ __forceinline__ uint2 ldg_list(const uint2 *p) {
    uint2 v;
    asm volatile("ld.global.nc.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p));
    return v;
}

// per-lane constants of the pair loop
template <typename real, int MODE>
struct LaneCtx {
    typename Vec4<real>::type pi;
    real gi;
    PairConsts<real> kc;
};
template <>
struct LaneCtx<float, MODE_TMU> {
    TmuLane L;
    TmuConsts K;
};

template <typename real, int MODE>
__device__ __forceinline__ void eval_quad(const unsigned char *s_base, int pay_stride, uint2 e,
                                          const LaneCtx<real, MODE> &lc, Partial<real, MODE> &A) {
    // two pairs at a time (two independent dependency chains; four measured slower: registers)
    const unsigned o0[2] = {e.x & 0xffffu, e.x >> 16}, o1[2] = {e.y & 0xffffu, e.y >> 16};
    eval_pairs<real, MODE, 2>(s_base, pay_stride, o0, lc.pi, lc.gi, lc.kc, A);
    eval_pairs<real, MODE, 2>(s_base, pay_stride, o1, lc.pi, lc.gi, lc.kc, A);
}
template <>
__device__ __forceinline__ void eval_quad<float, MODE_TMU>(const unsigned char *s_base, int pay_stride, uint2 e,
                                                           const LaneCtx<float, MODE_TMU> &lc,
                                                           Partial<float, MODE_TMU> &A) {
    tmu_pair2(s_base, pay_stride, e.x & 0xffffu, e.x >> 16, lc.L, lc.K, A);
    tmu_pair2(s_base, pay_stride, e.y & 0xffffu, e.y >> 16, lc.L, lc.K, A);
}

template <typename real, int MODE>
__device__ __forceinline__ void make_lane(LaneCtx<real, MODE> &lc, const typename Vec4<real>::type &pi, real gi,
                                          const PairConsts<real> &kc) {
    lc.pi = pi; lc.gi = gi; lc.kc = kc;
}
template <>
__device__ __forceinline__ void make_lane<float, MODE_TMU>(LaneCtx<float, MODE_TMU> &lc, const float4 &pi, float,
                                                           const PairConsts<float> &kc) {
    lc.L.pxy = pk(pi.x, pi.y);
    lc.L.nz0 = pk(-pi.z, 0.0f);
    lc.L.one_w = pk(1.0f, pi.w * 1.4426950408889634f);
    lc.K.pb = kc.pb;
    lc.K.nb2l = kc.nb2l;
    lc.K.c1b = kc.c1b;
    lc.K.k3 = kc.k3;
}

// trips of list rows (512 B per warp) the shared-memory ring holds; 0 = register prefetch
template <typename real, int MODE> struct ListRing { static constexpr int N = 0; };
template <> struct ListRing<float, MODE_TMU> { static constexpr int N = 4; };
constexpr int RING_ROW = 512;        // bytes per warp and trip

__device__ __forceinline__ void cp_async16(unsigned dst, const void *src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
template <int BYTES>
__device__ __forceinline__ void cp_async_rec(void *dst, const void *src) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst);
#pragma unroll
    for (int o = 0; o < BYTES; o += 16) cp_async16(d + o, reinterpret_cast<const unsigned char *>(src) + o);
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ uint4 lds128(unsigned addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
    return v;
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
    constexpr int SU = sizeof(real) == 8 ? 4 : 8;   // staged records in flight per thread
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
    // warps per block: a group with few blocks (small systems: config 1 has 1.7 blocks per group)
    // gives each block to 2, 4 or 8 warps; warp `part` of a block takes the block's list rows
    // part, part + wpb, ... and the parts are added in a fixed order at the end (bit-reproducible)
    const int wpb = nb >= 5 ? 1 : (nb >= 3 ? 2 : (nb == 2 ? 4 : 8));
    const int kb = w / wpb, part = w - kb * wpb;
    const bool active = kb < nb;
    const int blk = b0 + (active ? kb : 0);
    const int slot = blk * BLOCK + lane;
    const vec4 pi = gpos[slot];
    real gi = 0;
    if (MODE == MODE_FIELD) gi = data[2 * (size_t)n_pad + slot].z;
    const uint2 *__restrict__ lp = reinterpret_cast<const uint2 *>(ws.alist + (size_t)blk * ws.a_cap * 32) + lane * 2;
    const int32_t *__restrict__ arow = ws.arow + (size_t)blk * (NCH_MAX + 1);
    constexpr int RING = ListRing<real, MODE>::N;

    double dx = 0.0, dy = 0.0, dz = 0.0;
    Partial<real, MODE> A;
    LaneCtx<real, MODE> lc;
    make_lane<real, MODE>(lc, pi, gi, kc);
    int since_flush = 0;

    if (t == 0) {                              // permanent dummy record: far away, zero payload
        vec4 far, zero;
        far.x = far.y = far.z = (real)(-2.0f * PHANTOM_FAR); far.w = 0;
        zero.x = zero.y = zero.z = zero.w = 0;
        s_pos[s_chunk] = far;
        for (int k = 0; k < NPAY; ++k) s_pay[k * pstride + s_chunk] = zero;
    }

    // list ring (RING > 0): the block's rows are one contiguous stream over all chunks; this warp's
    // m-th row (row part + m wpb) goes to slot m % RING of its ring, RING - 1 trips before its use.
    // Every lane copies and reads only its own 16 bytes, so cp.async.wait_group is all the
    // synchronisation needed.
    const int t_total = (active && n_chunks <= NCH_MAX) ? arow[n_chunks] >> 3 : 0;
    const uint4 *const rows = reinterpret_cast<const uint4 *>(lp);          // row tg of this lane: rows[tg * 32]
    unsigned ring = 0;
    int t_issue = part, m_issue = 0, m_use = 0;
    if (RING > 0) {
        ring = (unsigned)__cvta_generic_to_shared(smem_raw) + (unsigned)((1 + NPAY) * pay_stride) +
               (unsigned)(w * RING * RING_ROW + lane * 16);
#pragma unroll
        for (int k = 0; k < RING - 1; ++k) {
            if (t_issue < t_total) cp_async16(ring + (m_issue % RING) * RING_ROW, rows + (size_t)t_issue * 32);
            cp_async_commit();
            t_issue += wpb; ++m_issue;
        }
    }

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
                if (idx < count) cp_async_rec<sizeof(vec4)>(s_pos + l0 + u * GT, stage_pos + gbase + idx);
            }
#pragma unroll
            for (int k = 0; k < NPAY; ++k) {
#pragma unroll
                for (int u = 0; u < SU; ++u)
                    if (a[u] >= 0) cp_async_rec<sizeof(vec4)>(s_pay + k * pstride + l0 + u * GT, data + (size_t)k * n_pad + a[u]);
            }
        }
        cp_async_commit();
        cp_async_wait<0>();
        __syncthreads();
        if (!active) continue;
        const int q0 = arow[c] >> 2, q1 = arow[c + 1] >> 2;
        if (q0 >= q1) continue;
        const unsigned char *s_base = smem_raw;
        if (RING > 0) {
            // my rows of this chunk: the smallest tg >= first row with tg = part (mod wpb)
            const int r0 = q0 >> 1;
            for (int tg = r0 + ((part - r0) & (wpb - 1)); tg < (q1 >> 1); tg += wpb) {
                if (t_issue < t_total) cp_async16(ring + (m_issue % RING) * RING_ROW, rows + (size_t)t_issue * 32);
                cp_async_commit();
                t_issue += wpb; ++m_issue;
                cp_async_wait<(RING > 0 ? RING - 1 : 0)>();
                const uint4 e = lds128(ring + (m_use % RING) * RING_ROW);
                ++m_use;
                eval_quad<real, MODE>(s_base, pay_stride, make_uint2(e.x, e.y), lc, A);
                eval_quad<real, MODE>(s_base, pay_stride, make_uint2(e.z, e.w), lc, A);
                if ((m_use & 3) == 0) A.flush(dx, dy, dz);   // every 32 entries: FP32 partial -> FP64
            }
        } else {
            // Two quads per trip; a quad is loaded one whole trip (8 pairs) before its use, right after
            // the registers it goes to have been unpacked.  The loads are volatile asm so that they
            // stay where they are written: a load that drifts to the end of the loop body shares its
            // scoreboard with the unpack at the top and exposes the full L2 latency in every trip.
            const int r0 = q0 >> 1;
            const int qf = (r0 + ((part - r0) & (wpb - 1))) << 1;  // first quad of my first row in this chunk
            if (qf >= q1) continue;
            const int qstep = 2 * wpb;
            const uint2 *pq = lp + qidx(qf);
            const uint2 *const pend = lp + qidx(qf + ((q1 - 2 - qf) / qstep) * qstep);   // my last row: clamp for the look-ahead loads
            const size_t pstep = (size_t)64 * wpb;
            uint2 eA = ldg_list(pq);
            uint2 eB = ldg_list(pq + 1);
            for (int q = qf; q < q1; q += qstep, pq += pstep) {
                const uint2 a = eA;
                eA = ldg_list(pq + pstep <= pend ? pq + pstep : pend);
                eval_quad<real, MODE>(s_base, pay_stride, a, lc, A);
                const uint2 b = eB;
                eB = ldg_list(pq + pstep <= pend ? pq + pstep + 1 : pend + 1);
                eval_quad<real, MODE>(s_base, pay_stride, b, lc, A);
                if (++since_flush == 4) {          // every 32 entries: FP32 partial -> FP64 accumulator
                    A.flush(dx, dy, dz);
                    since_flush = 0;
                }
            }
        }
    }
    if (RING > 0) cp_async_wait<0>();
    A.flush(dx, dy, dz);
    if (wpb > 1) {                             // uniform over the CTA: add the parts of a block, part 1 first
        double *s_part = reinterpret_cast<double *>(smem_raw);         // [warp][xyz][lane], over the dead records
        __syncthreads();
        if (part > 0) {
            s_part[w * 96 + lane] = dx; s_part[w * 96 + 32 + lane] = dy; s_part[w * 96 + 64 + lane] = dz;
        }
        __syncthreads();
        if (part == 0)
            for (int k = 1; k < wpb; ++k) {
                dx += s_part[(w + k) * 96 + lane]; dy += s_part[(w + k) * 96 + 32 + lane]; dz += s_part[(w + k) * 96 + 64 + lane];
            }
    }
    const bool owner = active && part == 0;
    if (owner) {
        acc[slot] = dx;
        acc[n_pad + slot] = dy;
        acc[2 * (size_t)n_pad + slot] = dz;
    }
    if (MODE == MODE_TMU && fuse.on) {
        double pq = 0, dummy = 0;
        if (owner) {
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
    const size_t smem = sizeof(vec4) * (size_t)(1 + NPAY) * (size_t)(s_chunk + 1) +
                        (size_t)ListRing<real, MODE>::N * RING_ROW * GB;
    static bool configured[2][2] = {{false, false}, {false, false}};
    if (!configured[which][MODE]) {
        TKHP_CUDA(c, cudaFuncSetAttribute(k_atom_pairs<real, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          2 * ATOM_SMEM + 4096 + ListRing<real, MODE>::N * RING_ROW * GB));
        configured[which][MODE] = true;
    }
    PairConsts<real> k;
    k.beta = (real)c->p.ewald_beta;
    k.c1 = (real)(2.0 / SQRT_PI);
    k.c23 = (real)(4.0 / (3.0 * SQRT_PI));
    k.rc2 = (real)(c->p.cutoff * c->p.cutoff);
    k.box = (real)1;
    k.inv_box = (real)0;
    {
        const double b = c->p.ewald_beta;
        k.pb = (real)((double)TKHP_ERFCX_P * b);
        k.nb2l = (real)(-1.4426950408889634 * b * b);
        k.c1b = (real)(2.0 / SQRT_PI * b);
        k.k3 = (real)(4.0 / (3.0 * SQRT_PI) * b * b * b);
    }
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
