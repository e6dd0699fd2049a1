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
        int qmax = (kmax + 3) >> 2;
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

// ----------------------------------------------------------------------------- pair kernels
//   MODE_TMU   (T1,T2): out_i += -m1 mu_j + m2 (mu_j.R) R            staged: pos+w, mu
//   MODE_FIELD (F1,F2): field at i from (q,d,Q)_j, same-group pairs contribute zero here (the FP64
//                       correction pass adds them, pcg.cu)            staged: pos+w, 3 multipole vec4
template <typename real, int MODE>
__device__ __forceinline__ void eval_pair2(const unsigned char *s_base, int pay_stride, unsigned o0, unsigned o1,
                                           const typename Vec4<real>::type &pi, real gi,
                                           const PairConsts<real> &kc, real &ax, real &ay, real &az) {
    using vec4 = typename Vec4<real>::type;
    constexpr int NK = MODE == MODE_TMU ? 2 : 3;
    const unsigned off[2] = {o0, o1};
    vec4 pj[2];
    real Rx[2], Ry[2], Rz[2], r2[2], ww[2], G[2][NK];
#pragma unroll
    for (int u = 0; u < 2; ++u) pj[u] = *reinterpret_cast<const vec4 *>(s_base + off[u]);
    if (MODE == MODE_TMU) {
        vec4 mj[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) mj[u] = *reinterpret_cast<const vec4 *>(s_base + pay_stride + off[u]);
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            Rx[u] = pi.x - pj[u].x; Ry[u] = pi.y - pj[u].y; Rz[u] = pi.z - pj[u].z;
            r2[u] = Rx[u] * Rx[u] + Ry[u] * Ry[u] + Rz[u] * Rz[u];
            ww[u] = pi.w * pj[u].w;
        }
        radial_w<NK, 2>(r2, ww, kc, G);
#pragma unroll
        for (int u = 0; u < 2; ++u)
            tmu_apply<real>(G[u][0], G[u][1], Rx[u], Ry[u], Rz[u], mj[u].x, mj[u].y, mj[u].z, ax, ay, az);
    } else {
        vec4 b0v[2], b1v[2], b2v[2];
        bool in[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            b0v[u] = *reinterpret_cast<const vec4 *>(s_base + pay_stride + off[u]);
            b1v[u] = *reinterpret_cast<const vec4 *>(s_base + 2 * pay_stride + off[u]);
            b2v[u] = *reinterpret_cast<const vec4 *>(s_base + 3 * pay_stride + off[u]);
        }
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            Rx[u] = pi.x - pj[u].x; Ry[u] = pi.y - pj[u].y; Rz[u] = pi.z - pj[u].z;
            r2[u] = Rx[u] * Rx[u] + Ry[u] * Ry[u] + Rz[u] * Rz[u];
            ww[u] = pi.w * pj[u].w;
            in[u] = b2v[u].z != gi;
        }
        radial_w<NK, 2>(r2, ww, kc, G);
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            if (!in[u]) { G[u][0] = 0; G[u][1] = 0; G[u][2] = 0; }
            field_apply<real>(G[u], Rx[u], Ry[u], Rz[u], b0v[u].x, b0v[u].y, b0v[u].z, b0v[u].w, b1v[u].x,
                              b1v[u].y, b1v[u].z, b1v[u].w, b2v[u].x, b2v[u].y, ax, ay, az);
        }
    }
}

template <typename real, int MODE>
__global__ void __launch_bounds__(GT)
k_atom_pairs(ClusterWs ws, const typename Vec4<real>::type *__restrict__ gpos,
             const typename Vec4<real>::type *__restrict__ stage_pos,
             const typename Vec4<real>::type *__restrict__ data,   // mu (n_pad) or multipoles (3 n_pad)
             PairConsts<real> kc, double *__restrict__ acc, int n_pad, int s_chunk,
             DeviceState *st, int iter, PcgFuse fuse) {
    if (iter >= 0 && iter >= st->conv_at) return;      // PCG already converged (pcg.cu)
    using vec4 = typename Vec4<real>::type;
    constexpr int NPAY = MODE == MODE_TMU ? 1 : 3;
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
        for (int l = t, idx = c + t * n_chunks; idx < count; l += GT, idx += GT * n_chunks) {
            const int a = ws.stage_atom[gbase + idx];
            s_pos[l] = stage_pos[gbase + idx];
#pragma unroll
            for (int k = 0; k < NPAY; ++k) s_pay[k * pstride + l] = data[(size_t)k * n_pad + a];
        }
        __syncthreads();
        if (!active) continue;
        const int q0 = arow[c] >> 2, q1 = arow[c + 1] >> 2;
        if (q0 >= q1) continue;
        const unsigned char *s_base = smem_raw;
        // list quads are fetched two steps ahead of their use (L2 latency under load ~ one step)
        uint2 e = lp[(size_t)q0 * 32];
        uint2 e1 = lp[(size_t)(q0 + 1 < q1 ? q0 + 1 : q0) * 32];
        for (int q = q0; q < q1; ++q) {
            const int qn = q + 2 < q1 ? q + 2 : q1 - 1;
            const uint2 e2 = lp[(size_t)qn * 32];
            eval_pair2<real, MODE>(s_base, pay_stride, e.x & 0xffffu, e.x >> 16, pi, gi, kc, ax, ay, az);
            eval_pair2<real, MODE>(s_base, pay_stride, e.y & 0xffffu, e.y >> 16, pi, gi, kc, ax, ay, az);
            e = e1;
            e1 = e2;
            if (++since_flush == 8) {          // every 32 entries: FP32 partial -> FP64 accumulator
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
    c->n_launches += 1;
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
