// cluster.cu -- CLUSTER list mode: filtered cluster->atom lists with the neighbourhood of a
// group of blocks staged in shared memory.
//
// Paper, "List filtering": "By filtering every neighboring group, we can get a list
// of atoms which really belong to a group's neighborhood ... alpha in B_I if there is alpha_i in
// beta_I such that dist(alpha_i, alpha) <= d_cut + d_buff ... phantom atoms to complete the actual
// neighbor lists ... a loss of coalesced memory access pattern ... compensated by an increase of
// B_comp", +75% on their vdW kernel, then applied to "electrostatics and polarization".
//
// B200 redesign:
//  * the filter granularity is an 8-atom CLUSTER (a quarter warp), not the 32-atom block: with
//    r_c = 7 A a 32-atom block is as wide as the cutoff and only ~26% of (block atom, list atom)
//    slots are inside r_c; for 8-atom clusters it is ~49% (measured, DESIGN.md table 5.1);
//  * the filter radius is r_c (+0.01 A guard), not r_c + skin: the list is used for the positions
//    it was built from (one solve), the skin only enters the prescribed block-pair list;
//  * a CTA owns a GROUP of up to 8 consecutive blocks; every list atom of the group's clusters is
//    staged ONCE in shared memory (position already shifted into the group's frame, so no image
//    arithmetic in the pair loop), and list entries are 16-bit indices into that staging area:
//    the "loss of coalesced access" the paper notes becomes conflict-free LDS.128 (each quarter
//    warp reads one 16-byte record, broadcast to its 8 lanes);
//  * every lane owns one atom i and only ever updates atom i: no atomics, no j-side accumulator,
//    bit-reproducible results; FP32 partials are flushed into FP64 registers every 32 entries
//    (64-bit containers for accumulation);
//  * the number of groups is a whole multiple of (SM count x resident CTAs) whenever the system
//    is smaller than a few waves, so every SM gets the same number of blocks.
#include "common.cuh"
#include "pair_math.cuh"

namespace tkhp {

constexpr int GB = 8;                 // max blocks per group (= warps per CTA)
constexpr int GT = GB * 32;           // threads per CTA
constexpr int OCT = GB * 4;           // clusters per group
constexpr int CB_CAP = 1024;          // candidate blocks per group
constexpr int RESIDENT = 3;           // CTAs per SM the group count is rounded to
constexpr int B200_SMS = 148;
constexpr float GUARD = 0.01f;        // list radius = r_c + GUARD (FP32 build arithmetic is safe)

struct ClusterWs {
    int n_groups, s_cap, l_cap;
    int32_t *group_first;             // n_groups + 1
    float4 *gpos32;                   // n_pad: atom in its group's frame (x,y,z,w)
    double4 *gpos64;
    int32_t *stage_count;             // n_groups
    int32_t *stage_atom;              // n_groups * s_cap: sorted slot of each staged atom
    float4 *stage_pos32;              // n_groups * s_cap: position in the group's frame (+w)
    double4 *stage_pos64;
    uint32_t *stage_mask;             // n_groups * s_cap: which clusters of the group list the atom
    uint16_t *entries;                // (n_pad/8) * l_cap
    int32_t *oct_len;                 // n_pad/8: padded list length (equal within a warp)
};

static int choose_groups(int n_blocks) {
    const int base = (n_blocks + GB - 1) / GB;
    const int wave = B200_SMS * RESIDENT;
    if (base >= 4 * wave) return base;
    int g = ((base + wave - 1) / wave) * wave;
    if (g > n_blocks) g = n_blocks;
    return g;
}

static void size_caps(const tkhp_params *p, int n_blocks, int *s_cap, int *l_cap) {
    const long long n_pad = (long long)n_blocks * BLOCK;
    long long s, l;
    if (p->box > 0.0) {
        const double rho = p->n_atoms / (p->box * p->box * p->box);
        const double e = 1.3 * cbrt(GT / rho);
        double edge = e + 2.0 * (p->cutoff + 1.0);
        if (edge > p->box) edge = p->box;
        s = (long long)(1.25 * edge * edge * edge * rho) + 64;
        const double r = p->cutoff + 3.0;
        l = (long long)(1.5 * 4.18879 * r * r * r * rho) + 64;
    } else {
        s = 8192;
        l = 2048;
    }
    if (p->max_nbrs_per_cluster > 0) l = p->max_nbrs_per_cluster;
    if (s > n_pad + 1) s = n_pad + 1;
    if (l > n_pad + 8) l = n_pad + 8;
    if (s > 65535) s = 65535;          // 16-bit entries
    *s_cap = (int)((s + 63) & ~63LL);
    *l_cap = (int)((l + 7) & ~7LL);
}

static size_t carve_cluster(const tkhp_params *p, int n_blocks, void *base, ClusterWs *out) {
    Carver w(base);
    ClusterWs ws;
    const size_t n_pad = (size_t)n_blocks * BLOCK;
    ws.n_groups = choose_groups(n_blocks);
    size_caps(p, n_blocks, &ws.s_cap, &ws.l_cap);
    const bool f64 = p->precision == TKHP_FP64;
    const size_t gs = (size_t)ws.n_groups * ws.s_cap;
    ws.group_first = w.take<int32_t>(ws.n_groups + 1);
    ws.gpos32 = w.take<float4>(n_pad);
    ws.gpos64 = f64 ? w.take<double4>(n_pad) : nullptr;
    ws.stage_count = w.take<int32_t>(ws.n_groups);
    ws.stage_atom = w.take<int32_t>(gs);
    ws.stage_pos32 = w.take<float4>(gs);
    ws.stage_pos64 = f64 ? w.take<double4>(gs) : nullptr;
    ws.stage_mask = w.take<uint32_t>(gs);
    ws.entries = w.take<uint16_t>((n_pad / CLUSTER) * ws.l_cap);
    ws.oct_len = w.take<int32_t>(n_pad / CLUSTER);
    w.take<char>(256);
    if (out) *out = ws;
    return w.off;
}

size_t cluster_workspace_bytes(const tkhp_params *p, int n_blocks) {
    if (p->list_mode != TKHP_LIST_CLUSTER) return 0;
    return carve_cluster(p, n_blocks, nullptr, nullptr);
}

static ClusterWs get_ws(Ctx *c) {
    ClusterWs ws;
    carve_cluster(&c->p, c->n_blocks, c->cl_ws, &ws);
    return ws;
}

// ----------------------------------------------------------------------------- build
__global__ void k_group_first(int32_t *group_first, int n_groups, int n_blocks) {
    int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g <= n_groups) group_first[g] = (int)(((long long)g * n_blocks) / n_groups);
}

__device__ __forceinline__ double gap2_boxes(const double *gc, const double *gh, const double4 &c,
                                             const double4 &h, double box) {
    double d[3] = {fabs(gc[0] - c.x), fabs(gc[1] - c.y), fabs(gc[2] - c.z)};
    const double hh[3] = {gh[0] + h.x, gh[1] + h.y, gh[2] + h.z};
    double s = 0.0;
    for (int k = 0; k < 3; ++k) {
        if (box > 0.0) d[k] = fmin(d[k], box - d[k]);
        const double g = fmax(0.0, d[k] - hh[k]);
        s += g * g;
    }
    return s;
}

__global__ void __launch_bounds__(GT)
k_cluster_build(ClusterWs ws, const float4 *__restrict__ xyzw32, const double4 *__restrict__ xyzw64,
                const double4 *__restrict__ bcentre, const double4 *__restrict__ bhalf,
                const double4 *__restrict__ scentre, const double4 *__restrict__ shalf, int n_blocks,
                int n_super, double box, double cutoff, DeviceState *st) {
    __shared__ float4 s_i[GT];
    __shared__ float s_olo[OCT][3], s_ohi[OCT][3];
    __shared__ int s_cand[CB_CAP];
    __shared__ int s_ncand;
    __shared__ double s_gc[3], s_gh[3];
    __shared__ int s_wsum[GB];
    __shared__ int s_base;

    const int g = blockIdx.x, t = threadIdx.x, lane = t & 31, w = t >> 5;
    const int b0 = ws.group_first[g], nb = ws.group_first[g + 1] - b0;
    const bool f64 = ws.gpos64 != nullptr;
    const double rcm = cutoff + (double)GUARD;
    const float rcm2 = (float)(rcm * rcm);

    // (a) group box = union of its block boxes
    if (t == 0) {
        double lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
        for (int b = b0; b < b0 + nb; ++b) {
            const double4 c = bcentre[b], h = bhalf[b];
            lo[0] = fmin(lo[0], c.x - h.x); hi[0] = fmax(hi[0], c.x + h.x);
            lo[1] = fmin(lo[1], c.y - h.y); hi[1] = fmax(hi[1], c.y + h.y);
            lo[2] = fmin(lo[2], c.z - h.z); hi[2] = fmax(hi[2], c.z + h.z);
        }
        double hmax = 0.0;
        for (int k = 0; k < 3; ++k) {
            s_gc[k] = 0.5 * (lo[k] + hi[k]);
            s_gh[k] = 0.5 * (hi[k] - lo[k]) + 1e-6;
            hmax = fmax(hmax, s_gh[k]);
        }
        // one image per staged atom is exact iff r_c + group half extent < box/2
        if (box > 0.0 && !(rcm + hmax < 0.5 * box)) st->cluster_bad = 1;
        s_ncand = 0;
        s_base = 0;
    }
    __syncthreads();
    const double gcx = s_gc[0], gcy = s_gc[1], gcz = s_gc[2];

    // (b) the group's own atoms in the group frame
    {
        float4 v = make_float4(PHANTOM_FAR * (2 + t), PHANTOM_FAR, PHANTOM_FAR, 0.f);
        if (w < nb) {
            const int blk = b0 + w, slot = blk * BLOCK + lane;
            const double4 c = bcentre[blk];
            const float4 p = xyzw32[slot];
            if (p.w > 0.f) {
                double x, y, z;
                if (f64) {
                    const double4 q = xyzw64[slot];
                    x = q.x + (c.x - gcx); y = q.y + (c.y - gcy); z = q.z + (c.z - gcz);
                    ws.gpos64[slot] = make_double4(x, y, z, q.w);
                } else {
                    x = (double)p.x + (c.x - gcx); y = (double)p.y + (c.y - gcy); z = (double)p.z + (c.z - gcz);
                }
                v = make_float4((float)x, (float)y, (float)z, p.w);
            } else if (f64) {
                ws.gpos64[slot] = make_double4(v.x, v.y, v.z, 0.0);
            }
            ws.gpos32[slot] = v;
        }
        s_i[t] = v;
    }
    __syncthreads();

    // (c) cluster boxes
    if (t < OCT) {
        float lo[3] = {3e38f, 3e38f, 3e38f}, hi[3] = {-3e38f, -3e38f, -3e38f};
        for (int a = 0; a < CLUSTER; ++a) {
            const float4 q = s_i[t * CLUSTER + a];
            if (q.w > 0.f) {
                lo[0] = fminf(lo[0], q.x); hi[0] = fmaxf(hi[0], q.x);
                lo[1] = fminf(lo[1], q.y); hi[1] = fmaxf(hi[1], q.y);
                lo[2] = fminf(lo[2], q.z); hi[2] = fmaxf(hi[2], q.z);
            }
        }
        for (int k = 0; k < 3; ++k) { s_olo[t][k] = lo[k]; s_ohi[t][k] = hi[k]; }
    }

    // (d) candidate blocks: warp 0 walks super-blocks, then blocks, in index order (deterministic)
    if (w == 0) {
        const double reach2 = rcm * rcm;
        int n = 0;
        for (int s0 = 0; s0 < n_super; s0 += 32) {
            const int sj = s0 + lane;
            bool cand = false;
            if (sj < n_super) cand = gap2_boxes(s_gc, s_gh, scentre[sj], shalf[sj], box) <= reach2;
            unsigned m = __ballot_sync(0xffffffffu, cand);
            while (m) {
                const int s = s0 + (__ffs(m) - 1);
                m &= m - 1;
                const int J = s * SUPER + lane;
                bool keep = false;
                if (J < n_blocks) keep = gap2_boxes(s_gc, s_gh, bcentre[J], bhalf[J], box) <= reach2;
                const unsigned km = __ballot_sync(0xffffffffu, keep);
                if (keep) {
                    const int pos = n + __popc(km & ((1u << lane) - 1u));
                    if (pos < CB_CAP) s_cand[pos] = J;
                }
                n += __popc(km);
            }
        }
        if (lane == 0) {
            if (n > CB_CAP) { st->cluster_bad = 1; n = CB_CAP; }
            s_ncand = n;
        }
    }
    __syncthreads();
    const int ncand = s_ncand;

    // (e) every atom of the candidate blocks against the group's clusters
    const size_t gbase = (size_t)g * ws.s_cap;
    for (int c0 = 0; c0 < ncand; c0 += GB) {
        uint32_t mask = 0;
        float4 pj = make_float4(0.f, 0.f, 0.f, 0.f);
        double px = 0, py = 0, pz = 0, pw = 0;
        int slot = -1;
        if (c0 + w < ncand) {
            const int J = s_cand[c0 + w];
            slot = J * BLOCK + lane;
            const float4 p = xyzw32[slot];
            if (p.w > 0.f) {
                const double4 cj = bcentre[J];
                double dx = cj.x - gcx, dy = cj.y - gcy, dz = cj.z - gcz;
                if (box > 0.0) {
                    dx -= box * rint(dx / box); dy -= box * rint(dy / box); dz -= box * rint(dz / box);
                }
                if (f64) {
                    const double4 q = xyzw64[slot];
                    px = q.x + dx; py = q.y + dy; pz = q.z + dz; pw = q.w;
                } else {
                    px = (double)p.x + dx; py = (double)p.y + dy; pz = (double)p.z + dz; pw = p.w;
                }
                pj = make_float4((float)px, (float)py, (float)pz, p.w);
                for (int o = 0; o < OCT; ++o) {
                    const float ex = fmaxf(0.f, fmaxf(s_olo[o][0] - pj.x, pj.x - s_ohi[o][0]));
                    const float ey = fmaxf(0.f, fmaxf(s_olo[o][1] - pj.y, pj.y - s_ohi[o][1]));
                    const float ez = fmaxf(0.f, fmaxf(s_olo[o][2] - pj.z, pj.z - s_ohi[o][2]));
                    if (ex * ex + ey * ey + ez * ez <= rcm2) {
                        bool any = false;
#pragma unroll
                        for (int a = 0; a < CLUSTER; ++a) {
                            const float4 q = s_i[o * CLUSTER + a];
                            const float ddx = q.x - pj.x, ddy = q.y - pj.y, ddz = q.z - pj.z;
                            any |= (ddx * ddx + ddy * ddy + ddz * ddz <= rcm2) && (q.w > 0.f);
                        }
                        if (any) mask |= 1u << o;
                    }
                }
            }
        }
        // block-wide exclusive rank of the staged atoms (warp ballots + 8 warp sums)
        const unsigned bal = __ballot_sync(0xffffffffu, mask != 0u);
        if (lane == 0) s_wsum[w] = __popc(bal);
        __syncthreads();
        int before = 0, total = 0;
        for (int k = 0; k < GB; ++k) {
            const int v = s_wsum[k];
            if (k < w) before += v;
            total += v;
        }
        const int base = s_base;
        if (mask != 0u) {
            const int idx = base + before + __popc(bal & ((1u << lane) - 1u));
            if (idx < ws.s_cap - 1) {
                ws.stage_atom[gbase + idx] = slot;
                ws.stage_pos32[gbase + idx] = pj;
                if (f64) ws.stage_pos64[gbase + idx] = make_double4(px, py, pz, pw);
                ws.stage_mask[gbase + idx] = mask;
            }
        }
        __syncthreads();
        if (t == 0) s_base = base + total;
        __syncthreads();
    }
    int count = s_base;
    if (count > ws.s_cap - 1) {
        if (t == 0) st->cluster_bad = 1;
        count = ws.s_cap - 1;
    }
    if (t == 0) {
        ws.stage_count[g] = count;
        atomicMax(&st->max_stage, count);
    }
    __syncthreads();

    // (f) per-cluster lists: entries are staging indices, in staging order
    if (w < nb) {
        int len[4];
        const int oct0 = (b0 + w) * 4;
        for (int oo = 0; oo < 4; ++oo) {
            const int o = w * 4 + oo;
            uint16_t *ent = ws.entries + (size_t)(oct0 + oo) * ws.l_cap;
            int n = 0;
            for (int base = 0; base < count; base += 32) {
                const int idx = base + lane;
                const bool bit = idx < count && ((ws.stage_mask[gbase + idx] >> o) & 1u);
                const unsigned bm = __ballot_sync(0xffffffffu, bit);
                if (bit) {
                    const int pos = n + __popc(bm & ((1u << lane) - 1u));
                    if (pos < ws.l_cap) ent[pos] = (uint16_t)idx;
                }
                n += __popc(bm);
            }
            len[oo] = n;
        }
        int L = max(max(len[0], len[1]), max(len[2], len[3]));
        if (L > ws.l_cap) {
            if (lane == 0) st->cluster_bad = 1;
            L = ws.l_cap;
        }
        L = (L + 7) & ~7;
        if (L > ws.l_cap) L = ws.l_cap;
        for (int oo = 0; oo < 4; ++oo) {
            uint16_t *ent = ws.entries + (size_t)(oct0 + oo) * ws.l_cap;
            for (int k = min(len[oo], L) + lane; k < L; k += 32) ent[k] = (uint16_t)count;   // dummy far atom
            if (lane == 0) ws.oct_len[oct0 + oo] = L;
        }
        if (lane == 0) atomicAdd((unsigned long long *)&st->n_cluster_entries, (unsigned long long)(4 * L));
    }
}

// ----------------------------------------------------------------------------- T.mu
template <typename real>
__global__ void __launch_bounds__(GT)
k_cluster_tmu(ClusterWs ws, const typename Vec4<real>::type *__restrict__ gpos,
              const typename Vec4<real>::type *__restrict__ stage_pos,
              const typename Vec4<real>::type *__restrict__ mu, PairConsts<real> kc,
              double *__restrict__ acc, int n_pad, int s_run) {
    using vec4 = typename Vec4<real>::type;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    vec4 *s_pos = reinterpret_cast<vec4 *>(smem_raw);
    vec4 *s_mu = s_pos + s_run;

    const int g = blockIdx.x, t = threadIdx.x, lane = t & 31, w = t >> 5;
    const int b0 = ws.group_first[g], nb = ws.group_first[g + 1] - b0;
    const int count = ws.stage_count[g];
    const size_t gbase = (size_t)g * ws.s_cap;
    for (int idx = t; idx < count; idx += GT) {
        s_pos[idx] = stage_pos[gbase + idx];
        s_mu[idx] = mu[ws.stage_atom[gbase + idx]];
    }
    if (t == 0) {
        vec4 far, zero;
        far.x = far.y = far.z = (real)(-2.0f * PHANTOM_FAR); far.w = 0;
        zero.x = zero.y = zero.z = zero.w = 0;
        s_pos[count] = far;
        s_mu[count] = zero;
    }
    __syncthreads();
    if (w >= nb) return;

    const int slot = (b0 + w) * BLOCK + lane;
    const vec4 pi = gpos[slot];
    const int oct = slot >> 3;
    const int L = ws.oct_len[oct];
    const uint16_t *__restrict__ ent = ws.entries + (size_t)oct * ws.l_cap;
    const int qbase = lane & 24;
    double dx = 0.0, dy = 0.0, dz = 0.0;
    real ax = 0, ay = 0, az = 0;
    for (int k0 = 0; k0 < L; k0 += 8) {
        const unsigned e = ent[k0 + (lane & 7)];
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) {
            const unsigned idx = __shfl_sync(0xffffffffu, e, qbase + kk);
            const vec4 pj = s_pos[idx];
            const vec4 mj = s_mu[idx];
            const real Rx = pi.x - pj.x, Ry = pi.y - pj.y, Rz = pi.z - pj.z;
            const real r2 = Rx * Rx + Ry * Ry + Rz * Rz;
            const bool in = (r2 <= kc.rc2) && (r2 > (real)1e-10);
            real G[2];
            radial<2>(in ? r2 : (real)1, pi.w * pj.w, kc, G);
            const real m1 = in ? G[0] : (real)0, m2 = in ? G[1] : (real)0;
            tmu_apply<real>(m1, m2, Rx, Ry, Rz, mj.x, mj.y, mj.z, ax, ay, az);
        }
        if ((k0 & 24) == 24) {   // every 32 entries: FP32 partial -> FP64 accumulator
            dx += (double)ax; dy += (double)ay; dz += (double)az;
            ax = 0; ay = 0; az = 0;
        }
    }
    dx += (double)ax; dy += (double)ay; dz += (double)az;
    acc[slot] = dx;
    acc[n_pad + slot] = dy;
    acc[2 * (size_t)n_pad + slot] = dz;
}

// ----------------------------------------------------------------------------- host side
int cluster_build(Ctx *c, cudaStream_t s) {
    ClusterWs ws = get_ws(c);
    k_group_first<<<div_up(ws.n_groups + 1, 256), 256, 0, s>>>(ws.group_first, ws.n_groups, c->n_blocks);
    k_cluster_build<<<ws.n_groups, GT, 0, s>>>(ws, c->xyzw32, c->xyzw64, c->bcentre, c->bhalf, c->scentre,
                                               c->shalf, c->n_blocks, c->n_super, c->p.box, c->p.cutoff, c->st);
    c->n_launches += 2;
    TKHP_CUDA(c, cudaGetLastError());
    return TKHP_OK;
}

template <typename real>
static int launch_tmu(Ctx *c, const ClusterWs &ws, cudaStream_t s) {
    using vec4 = typename Vec4<real>::type;
    const int s_run = ((c->h_state->max_stage + 1) + 15) & ~15;
    const size_t smem = 2 * sizeof(vec4) * (size_t)s_run;
    if (smem > 227 * 1024) return set_err(c, TKHP_ECAPACITY, "cluster staging exceeds shared memory%s");
    static size_t configured[2] = {0, 0};
    const int which = sizeof(real) == 8;
    if (smem > configured[which]) {
        TKHP_CUDA(c, cudaFuncSetAttribute(k_cluster_tmu<real>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(227 * 1024)));
        configured[which] = 227 * 1024;
    }
    PairConsts<real> k;
    k.beta = (real)c->p.ewald_beta;
    k.c1 = (real)(2.0 / SQRT_PI);
    k.rc2 = (real)(c->p.cutoff * c->p.cutoff);
    k.box = (real)1; k.inv_box = (real)0;
    const vec4 *gpos = which ? (const vec4 *)ws.gpos64 : (const vec4 *)ws.gpos32;
    const vec4 *spos = which ? (const vec4 *)ws.stage_pos64 : (const vec4 *)ws.stage_pos32;
    const vec4 *mu = which ? (const vec4 *)c->mu64 : (const vec4 *)c->mu32;
    k_cluster_tmu<real><<<ws.n_groups, GT, smem, s>>>(ws, gpos, spos, mu, k, c->acc, c->n_pad, s_run);
    c->n_launches += 1;
    TKHP_CUDA(c, cudaGetLastError());
    return TKHP_OK;
}

int cluster_tmatvec(Ctx *c, cudaStream_t s) {
    ClusterWs ws = get_ws(c);
    return c->p.precision == TKHP_MIXED ? launch_tmu<float>(c, ws, s) : launch_tmu<double>(c, ws, s);
}

int cluster_field(Ctx *c, cudaStream_t s) {
    // the permanent field runs once per solve: it walks the block-pair list (tiles.cu);
    // run_field() has zeroed the accumulators
    return tiles_field(c, s);
}

long long cluster_slots(Ctx *c) { return 8LL * c->h_state->n_cluster_entries; }

}  // namespace tkhp
