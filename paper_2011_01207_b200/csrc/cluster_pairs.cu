// cluster_pairs.cu -- the pair kernels of CLUSTER list mode (design: cluster.cuh).
//
// One CTA per group of <= 8 blocks; warp w owns block b0 + w, lane l owns atom i = 32 (b0+w) + l.
// A quarter warp (8 lanes) is one cluster and walks its own list: per step all 8 lanes read the
// SAME staged atom j (one conflict-free LDS.128 per record and quarter warp) and each evaluates
// its pair (i, j) in one direction: atom i only.  The staging area holds a CHUNK of the group's
// staged atoms (lists are in staging order, so each cluster consumes a prefix of its remaining
// entries per chunk); one chunk is the common case, more chunks bound the shared memory per CTA
// for FP64, the field kernel and long cutoffs, which keeps 3 CTAs resident per SM.
// The next 8 list entries are fetched while the current 8 are evaluated, and pairs are evaluated
// two at a time (W = 2 independent dependency chains per lane).
//
//   MODE_TMU   (T1,T2): out_i += -m1 mu_j + m2 (mu_j.R) R            staged: pos+w, mu
//   MODE_FIELD (F1,F2): field at i from (q,d,Q)_j, same-group pairs skipped (FP64 correction
//                       pass adds them, pcg.cu)                       staged: pos+w, 3 multipole vec4
#include "cluster.cuh"

namespace tkhp {

constexpr int MODE_TMU = 0, MODE_FIELD = 1;
constexpr int SMEM_BUDGET = 72 * 1024;   // per CTA: 3 CTAs per SM
constexpr int W = 2;                     // pairs evaluated together per lane

template <typename real, int MODE>
__global__ void __launch_bounds__(GT)
k_cluster_pairs(ClusterWs ws, const typename Vec4<real>::type *__restrict__ gpos,
                const typename Vec4<real>::type *__restrict__ stage_pos,
                const typename Vec4<real>::type *__restrict__ data,   // mu (n_pad) or multipoles (3 n_pad)
                PairConsts<real> kc, double *__restrict__ acc, int n_pad, int s_chunk,
                const DeviceState *__restrict__ st, int iter) {
    if (iter >= 0 && iter >= st->conv_at) return;      // PCG already converged (pcg.cu)
    using vec4 = typename Vec4<real>::type;
    constexpr int NPAY = MODE == MODE_TMU ? 1 : 3;
    constexpr int NK = MODE == MODE_TMU ? 2 : 3;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    vec4 *s_pos = reinterpret_cast<vec4 *>(smem_raw);          // [s_chunk + 1], last = dummy
    vec4 *s_pay = s_pos + (s_chunk + 1);                       // NPAY arrays of [s_chunk + 1]
    const int pstride = s_chunk + 1;

    const int g = blockIdx.x, t = threadIdx.x, lane = t & 31, w = t >> 5;
    const int b0 = ws.group_first[g], nb = ws.group_first[g + 1] - b0;
    const int count = ws.stage_count[g];
    const size_t gbase = (size_t)g * ws.s_cap;
    const bool active = w < nb;

    const int slot = (b0 + (active ? w : 0)) * BLOCK + lane;
    const vec4 pi = gpos[slot];
    real gi = 0;
    if (MODE == MODE_FIELD) gi = data[2 * (size_t)n_pad + slot].z;
    const int oct = slot >> 3;
    const int L = active ? ws.oct_len[oct] : 0;
    const uint16_t *__restrict__ ent = ws.entries + (size_t)oct * ws.l_cap;
    const int qbase = lane & 24, ql = lane & 7;
    int cur = 0;                               // this cluster's cursor into its list
    double dx = 0.0, dy = 0.0, dz = 0.0;
    real ax = 0, ay = 0, az = 0;
    int since_flush = 0;
    const bool fixed = sizeof(real) == 4 && kc.fixed != 0;
    unsigned e = ql < L ? (unsigned)ent[ql] : 0xffffffffu;     // entries [cur, cur+8) of this cluster

    if (t == 0) {                              // permanent dummy record: far away, zero payload
        vec4 far, zero;
        far.x = far.y = far.z = (real)(-2.0f * PHANTOM_FAR); far.w = 0;
        zero.x = zero.y = zero.z = zero.w = 0;
        s_pos[s_chunk] = far;
        for (int k = 0; k < NPAY; ++k) s_pay[k * pstride + s_chunk] = zero;
    }

    // the dummy entry value `count` is processed in the last chunk (maps to the dummy record)
    for (int c0 = 0; c0 <= count; c0 += s_chunk) {
        const int c1 = min(c0 + s_chunk, count);          // staged atoms [c0, c1) live in this chunk
        __syncthreads();
        for (int idx = c0 + t; idx < c1; idx += GT) {
            const int a = ws.stage_atom[gbase + idx];
            s_pos[idx - c0] = stage_pos[gbase + idx];
#pragma unroll
            for (int k = 0; k < NPAY; ++k) s_pay[k * pstride + (idx - c0)] = data[(size_t)k * n_pad + a];
        }
        __syncthreads();
        const bool last = c0 + s_chunk > count;
        const int end = last ? 0x7fffffff : c1;           // entries below `end` belong to this chunk
        if (!active) continue;
        for (;;) {
            const bool ok = e != 0xffffffffu && (int)e < end;
            const unsigned okm = __ballot_sync(0xffffffffu, ok);
            if (okm == 0u) break;
            const int n_ok = __popc((okm >> qbase) & 0xffu);   // sorted list: a prefix is valid
            const unsigned loc = ok ? (e >= (unsigned)count ? (unsigned)s_chunk : e - (unsigned)c0)
                                    : (unsigned)s_chunk;
            // prefetch this cluster's next 8 entries (they are consumed ~500 instructions later)
            cur += n_ok;
            const int kn = cur + ql;
            const unsigned e_next = kn < L ? (unsigned)ent[kn] : 0xffffffffu;
#pragma unroll
            for (int kk = 0; kk < 8; kk += W) {
                vec4 pj[W];
                real Rx[W], Ry[W], Rz[W], r2[W], r2s[W], ww[W], G[W][NK];
                bool in[W];
                unsigned idx[W];
#pragma unroll
                for (int u = 0; u < W; ++u) idx[u] = __shfl_sync(0xffffffffu, loc, qbase + kk + u);
#pragma unroll
                for (int u = 0; u < W; ++u) pj[u] = s_pos[idx[u]];
#pragma unroll
                for (int u = 0; u < W; ++u) {
                    Rx[u] = pi.x - pj[u].x; Ry[u] = pi.y - pj[u].y; Rz[u] = pi.z - pj[u].z;
                    r2[u] = Rx[u] * Rx[u] + Ry[u] * Ry[u] + Rz[u] * Rz[u];
                    in[u] = (r2[u] <= kc.rc2) && (r2[u] > (real)1e-10);
                    r2s[u] = in[u] ? r2[u] : (real)1;
                    ww[u] = pi.w * pj[u].w;
                }
                if (MODE == MODE_TMU) {
                    vec4 mj[W];
#pragma unroll
                    for (int u = 0; u < W; ++u) mj[u] = s_pay[idx[u]];
                    radial_w<NK, W>(r2s, ww, kc, G);
#pragma unroll
                    for (int u = 0; u < W; ++u) {
                        const real m1 = in[u] ? G[u][0] : (real)0, m2 = in[u] ? G[u][1] : (real)0;
                        tmu_apply<real>(m1, m2, Rx[u], Ry[u], Rz[u], mj[u].x, mj[u].y, mj[u].z, ax, ay, az);
                    }
                } else {
                    vec4 b0v[W], b1v[W], b2v[W];
#pragma unroll
                    for (int u = 0; u < W; ++u) {
                        b0v[u] = s_pay[idx[u]];
                        b1v[u] = s_pay[pstride + idx[u]];
                        b2v[u] = s_pay[2 * pstride + idx[u]];
                        in[u] = in[u] && (b2v[u].z != gi);
                        r2s[u] = in[u] ? r2[u] : (real)1;
                    }
                    radial_w<NK, W>(r2s, ww, kc, G);
#pragma unroll
                    for (int u = 0; u < W; ++u) {
                        if (!in[u]) { G[u][0] = 0; G[u][1] = 0; G[u][2] = 0; }
                        field_apply<real>(G[u], Rx[u], Ry[u], Rz[u], b0v[u].x, b0v[u].y, b0v[u].z, b0v[u].w,
                                          b1v[u].x, b1v[u].y, b1v[u].z, b1v[u].w, b2v[u].x, b2v[u].y, ax, ay, az);
                    }
                }
            }
            e = e_next;
            if (++since_flush == 4) {          // every 32 entries: FP32 partial -> 64-bit container
                acc_add(dx, ax, fixed); acc_add(dy, ay, fixed); acc_add(dz, az, fixed);
                ax = 0; ay = 0; az = 0;
                since_flush = 0;
            }
        }
    }
    if (!active) return;
    acc_add(dx, ax, fixed); acc_add(dy, ay, fixed); acc_add(dz, az, fixed);
    acc[slot] = acc_value(dx, fixed);
    acc[n_pad + slot] = acc_value(dy, fixed);
    acc[2 * (size_t)n_pad + slot] = acc_value(dz, fixed);
}

template <typename real, int MODE>
static int launch_pairs(Ctx *c, const ClusterWs &ws, cudaStream_t s) {
    using vec4 = typename Vec4<real>::type;
    constexpr int NPAY = MODE == MODE_TMU ? 1 : 3;
    const size_t per = sizeof(vec4) * (1 + NPAY);
    int s_chunk = (int)(SMEM_BUDGET / per) - 1;
    const int need = c->h_state->max_stage + 1;
    if (need < s_chunk) s_chunk = need;
    if (s_chunk < 32) s_chunk = 32;
    const size_t smem = per * (size_t)(s_chunk + 1);
    const int which = sizeof(real) == 8;
    PairConsts<real> k = {};
    k.beta = (real)c->p.ewald_beta;
    k.c1 = (real)(2.0 / SQRT_PI);
    k.c23 = (real)(4.0 / (3.0 * SQRT_PI));
    k.rc2 = (real)(c->p.cutoff * c->p.cutoff);
    k.box = (real)1;
    k.inv_box = (real)0;
    k.fixed = c->fixed ? 1 : 0;
    const vec4 *gpos = which ? (const vec4 *)ws.gpos64 : (const vec4 *)ws.gpos32;
    const vec4 *spos = which ? (const vec4 *)ws.stage_pos64 : (const vec4 *)ws.stage_pos32;
    const vec4 *data;
    if (MODE == MODE_TMU) data = which ? (const vec4 *)c->mu64 : (const vec4 *)c->mu32;
    else data = which ? (const vec4 *)c->mp64 : (const vec4 *)c->mp32;
    k_cluster_pairs<real, MODE><<<ws.n_groups, GT, smem, s>>>(ws, gpos, spos, data, k, c->acc, c->n_pad, s_chunk, c->st, c->spec_iter);
    c->n_launches += 1;
    TKHP_CUDA(c, cudaGetLastError());
    return TKHP_OK;
}

// dynamic shared memory opt-in, once per context (the attribute is per device)
int cluster_pairs_configure(Ctx *c) {
    TKHP_CUDA(c, cudaFuncSetAttribute(k_cluster_pairs<float, MODE_TMU>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BUDGET + 1024));
    TKHP_CUDA(c, cudaFuncSetAttribute(k_cluster_pairs<float, MODE_FIELD>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BUDGET + 1024));
    TKHP_CUDA(c, cudaFuncSetAttribute(k_cluster_pairs<double, MODE_TMU>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BUDGET + 1024));
    TKHP_CUDA(c, cudaFuncSetAttribute(k_cluster_pairs<double, MODE_FIELD>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BUDGET + 1024));
    return TKHP_OK;
}

int cluster_tmatvec(Ctx *c, cudaStream_t s) {
    ClusterWs ws = get_ws(c);
    return c->p.precision != TKHP_FP64 ? launch_pairs<float, MODE_TMU>(c, ws, s)
                                        : launch_pairs<double, MODE_TMU>(c, ws, s);
}

int cluster_field(Ctx *c, cudaStream_t s) {
    ClusterWs ws = get_ws(c);
    return c->p.precision != TKHP_FP64 ? launch_pairs<float, MODE_FIELD>(c, ws, s)
                                        : launch_pairs<double, MODE_FIELD>(c, ws, s);
}

}  // namespace tkhp
