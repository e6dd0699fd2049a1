// cluster_build.cu -- construction of the CLUSTER lists (see cluster.cuh for the design).
#include "cluster.cuh"

namespace tkhp {

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
    __shared__ float4 s_i[GT + OCT];      // atom a of cluster o at o * 9 + a: lanes that read different clusters hit different bank groups
    __shared__ float s_olo[OCT][3], s_ohi[OCT][3];
    __shared__ int s_cand[CB_CAP];
    __shared__ int s_ncand;
    __shared__ double s_gc[3], s_gh[3];
    __shared__ int s_wsum[GB];
    __shared__ int s_base;
    __shared__ float4 s_q[2 * GT];        // (e): queue of candidate atoms that passed the group-box test
    __shared__ int s_qslot[2 * GT];

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
        s_i[(t >> 3) * 9 + (t & 7)] = v;
    }
    __syncthreads();

    // (c) cluster boxes
    if (t < OCT) {
        float lo[3] = {3e38f, 3e38f, 3e38f}, hi[3] = {-3e38f, -3e38f, -3e38f};
        for (int a = 0; a < CLUSTER; ++a) {
            const float4 q = s_i[t * 9 + a];
            if (q.w > 0.f) {
                lo[0] = fminf(lo[0], q.x); hi[0] = fmaxf(hi[0], q.x);
                lo[1] = fminf(lo[1], q.y); hi[1] = fmaxf(hi[1], q.y);
                lo[2] = fminf(lo[2], q.z); hi[2] = fmaxf(hi[2], q.z);
            }
        }
        for (int k = 0; k < 3; ++k) { s_olo[t][k] = lo[k]; s_ohi[t][k] = hi[k]; }
    }

    // (d) candidate blocks: in every round of 256 super-blocks warp w takes 32 consecutive ones (one
    // per lane), then the blocks of its hits; the warps' hits are concatenated in warp order, i.e.
    // in block index order (deterministic).
    {
        const double reach2 = rcm * rcm;
        int n = 0;                                   // candidates found so far (uniform over the CTA)
        for (int s0 = 0; s0 < n_super; s0 += GB * 32) {
            // one super-block per lane: 32 consecutive super-blocks per warp
            const int sj = s0 + w * 32 + lane;
            bool cand = false;
            if (sj < n_super) cand = gap2_boxes(s_gc, s_gh, scentre[sj], shalf[sj], box) <= reach2;
            unsigned m = __ballot_sync(0xffffffffu, cand);
            // two passes over the warp's candidate super-blocks: count, then write at the warp's offset
            int mine = 0;
            unsigned mm = m;
            while (mm) {
                const int sb = s0 + w * 32 + (__ffs(mm) - 1);
                mm &= mm - 1;
                const int J = sb * SUPER + lane;
                bool keep = false;
                if (J < n_blocks) keep = gap2_boxes(s_gc, s_gh, bcentre[J], bhalf[J], box) <= reach2;
                mine += __popc(__ballot_sync(0xffffffffu, keep));
            }
            if (lane == 0) s_wsum[w] = mine;
            __syncthreads();
            int before = 0, total = 0;
            for (int k = 0; k < GB; ++k) {
                const int v = s_wsum[k];
                if (k < w) before += v;
                total += v;
            }
            int pos0 = n + before;
            mm = m;
            while (mm) {
                const int sb = s0 + w * 32 + (__ffs(mm) - 1);
                mm &= mm - 1;
                const int J = sb * SUPER + lane;
                bool keep = false;
                if (J < n_blocks) keep = gap2_boxes(s_gc, s_gh, bcentre[J], bhalf[J], box) <= reach2;
                const unsigned km = __ballot_sync(0xffffffffu, keep);
                if (keep) {
                    const int pos = pos0 + __popc(km & ((1u << lane) - 1u));
                    if (pos < CB_CAP) s_cand[pos] = J;
                }
                pos0 += __popc(km);
            }
            n += total;
            __syncthreads();
        }
        if (t == 0) {
            if (n > CB_CAP) { st->cluster_bad = 1; n = CB_CAP; }
            s_ncand = n;
        }
    }
    __syncthreads();
    const int ncand = s_ncand;

    // (e) every atom of the candidate blocks against the group's clusters, in two steps.  Step 1 (cheap,
    // one candidate block per warp): the atom's image in the group frame and a test against the GROUP box;
    // the survivors (about half of the candidate atoms) are appended, in candidate order, to a queue in
    // shared memory.  Step 2 (expensive, whenever the queue holds a full CTA of atoms): one queued atom
    // per thread against the 32 cluster boxes, then against the atoms of the clusters within reach.  All
    // lanes of step 2 have work, and the staging order is the candidate order, as before.
    const size_t gbase = (size_t)g * ws.s_cap;
    const float ghx = (float)s_gh[0] + 1e-4f, ghy = (float)s_gh[1] + 1e-4f, ghz = (float)s_gh[2] + 1e-4f;
    const float rcm2_loose = rcm2 * 1.0001f;
    int q_n = 0;                                       // queued atoms (uniform over the CTA)
    for (int c0 = 0; c0 < ncand || q_n > 0; c0 += GB) {
        // ---- step 1
        if (c0 < ncand) {
            bool keep = false;
            float4 pj = make_float4(0.f, 0.f, 0.f, 0.f);
            int slot = -1;
            if (c0 + w < ncand) {
                const int J = s_cand[c0 + w];
                slot = J * BLOCK + lane;
                const float4 p = xyzw32[slot];
                if (p.w > 0.f) {
                    const double4 cj = bcentre[J];
                    double px = (double)p.x + (cj.x - gcx), py = (double)p.y + (cj.y - gcy), pz = (double)p.z + (cj.z - gcz);
                    if (f64) {
                        const double4 q = xyzw64[slot];
                        px = q.x + (cj.x - gcx); py = q.y + (cj.y - gcy); pz = q.z + (cj.z - gcz);
                    }
                    // the image is chosen per ATOM (unique because r_c + group half extent < box/2);
                    // a per-block shift would be ambiguous when r_c + both extents exceeds box/2
                    if (box > 0.0) {
                        px -= box * rint(px / box); py -= box * rint(py / box); pz -= box * rint(pz / box);
                    }
                    pj = make_float4((float)px, (float)py, (float)pz, p.w);
                    const float ex = fmaxf(0.f, fabsf(pj.x) - ghx), ey = fmaxf(0.f, fabsf(pj.y) - ghy), ez = fmaxf(0.f, fabsf(pj.z) - ghz);
                    keep = ex * ex + ey * ey + ez * ez <= rcm2_loose;
                }
            }
            const unsigned bal = __ballot_sync(0xffffffffu, keep);
            if (lane == 0) s_wsum[w] = __popc(bal);
            __syncthreads();
            int before = 0, total = 0;
            for (int k = 0; k < GB; ++k) {
                const int v = s_wsum[k];
                if (k < w) before += v;
                total += v;
            }
            if (keep) {
                const int pos = q_n + before + __popc(bal & ((1u << lane) - 1u));
                s_q[pos] = pj;
                s_qslot[pos] = slot;
            }
            q_n += total;
            __syncthreads();
            if (q_n < GT && c0 + GB < ncand) continue;          // wait for a full CTA of queued atoms
        }
        // ---- step 2: the first min(GT, q_n) queued atoms
        const int n_now = min(GT, q_n);
        uint32_t mask = 0;
        float4 pj = make_float4(0.f, 0.f, 0.f, 0.f);
        int slot = -1;
        if (t < n_now) {
            pj = s_q[t];
            slot = s_qslot[t];
            // first the 32 cluster boxes (uniform loop), then the atoms of the clusters whose box
            // is within reach (a loop over the set bits: ~1/4 of the clusters)
            uint32_t near_box = 0;
#pragma unroll 8
            for (int o = 0; o < OCT; ++o) {
                const float ex = fmaxf(0.f, fmaxf(s_olo[o][0] - pj.x, pj.x - s_ohi[o][0]));
                const float ey = fmaxf(0.f, fmaxf(s_olo[o][1] - pj.y, pj.y - s_ohi[o][1]));
                const float ez = fmaxf(0.f, fmaxf(s_olo[o][2] - pj.z, pj.z - s_ohi[o][2]));
                if (ex * ex + ey * ey + ez * ez <= rcm2) near_box |= 1u << o;
            }
            while (near_box) {
                const int o = __ffs(near_box) - 1;
                near_box &= near_box - 1;
                // (phantom atoms sit at PHANTOM_FAR: no test of w needed); two halves: most clusters whose
                // box is within reach have an atom within reach among the first four
                bool any = false;
#pragma unroll
                for (int a = 0; a < CLUSTER / 2; ++a) {
                    const float4 q = s_i[o * 9 + a];
                    const float ddx = q.x - pj.x, ddy = q.y - pj.y, ddz = q.z - pj.z;
                    any |= ddx * ddx + ddy * ddy + ddz * ddz <= rcm2;
                }
                if (!any) {
#pragma unroll
                    for (int a = CLUSTER / 2; a < CLUSTER; ++a) {
                        const float4 q = s_i[o * 9 + a];
                        const float ddx = q.x - pj.x, ddy = q.y - pj.y, ddz = q.z - pj.z;
                        any |= ddx * ddx + ddy * ddy + ddz * ddz <= rcm2;
                    }
                }
                if (any) mask |= 1u << o;
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
                if (f64) {
                    // the FP64 image again (same arithmetic as step 1)
                    const int J = slot / BLOCK;
                    const double4 cj = bcentre[J];
                    const double4 q = xyzw64[slot];
                    double px = q.x + (cj.x - gcx), py = q.y + (cj.y - gcy), pz = q.z + (cj.z - gcz);
                    if (box > 0.0) {
                        px -= box * rint(px / box); py -= box * rint(py / box); pz -= box * rint(pz / box);
                    }
                    ws.stage_pos64[gbase + idx] = make_double4(px, py, pz, q.w);
                }
                ws.stage_mask[gbase + idx] = mask;
            }
        }
        // the rest of the queue moves to the front
        float4 mv = make_float4(0.f, 0.f, 0.f, 0.f);
        int mvs = -1;
        if (GT + t < q_n) { mv = s_q[GT + t]; mvs = s_qslot[GT + t]; }
        __syncthreads();
        if (t == 0) s_base = base + total;
        if (GT + t < q_n) { s_q[t] = mv; s_qslot[t] = mvs; }
        q_n -= n_now;
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
        int len[4] = {0, 0, 0, 0};
        const int oct0 = (b0 + w) * 4;
        uint16_t *ent[4];
        for (int oo = 0; oo < 4; ++oo) ent[oo] = ws.entries + (size_t)(oct0 + oo) * ws.l_cap;
        // one pass over the staged atoms for the warp's 4 clusters; the mask of the next round is
        // loaded before the ballots of this one
        uint32_t m_next = lane < count ? ws.stage_mask[gbase + lane] : 0u;
        for (int base = 0; base < count; base += 32) {
            const int idx = base + lane;
            const uint32_t m = (m_next >> (w * 4)) & 0xfu;
            m_next = idx + 32 < count ? ws.stage_mask[gbase + idx + 32] : 0u;
#pragma unroll
            for (int oo = 0; oo < 4; ++oo) {
                const bool bit = (m >> oo) & 1u;
                const unsigned bm = __ballot_sync(0xffffffffu, bit);
                if (bit) {
                    const int pos = len[oo] + __popc(bm & ((1u << lane) - 1u));
                    if (pos < ws.l_cap) ent[oo][pos] = (uint16_t)idx;
                }
                len[oo] += __popc(bm);
            }
        }
        int L = max(max(len[0], len[1]), max(len[2], len[3]));
        if (L > ws.l_cap) {
            if (lane == 0) st->cluster_bad = 1;
            L = ws.l_cap;
        }
        L = (L + 7) & ~7;
        if (L > ws.l_cap) L = ws.l_cap;
        for (int oo = 0; oo < 4; ++oo) {
            for (int k = min(len[oo], L) + lane; k < L; k += 32) ent[oo][k] = (uint16_t)count;   // dummy far atom
            if (lane == 0) ws.oct_len[oct0 + oo] = L;
        }
        if (lane == 0) atomicAdd((unsigned long long *)&st->n_cluster_entries, (unsigned long long)(4 * L));
    }
}

size_t cluster_workspace_bytes(const tkhp_params *p, int n_blocks) {
    if (p->list_mode == TKHP_LIST_TILES) return 0;
    return carve_cluster(p, n_blocks, nullptr, nullptr);
}

int cluster_build(Ctx *c, cudaStream_t s) {
    ClusterWs ws = get_ws(c);
    k_cluster_build<<<ws.n_groups, GT, 0, s>>>(ws, c->xyzw32, c->xyzw64, c->bcentre, c->bhalf, c->scentre,
                                               c->shalf, c->n_blocks, c->n_super, c->p.box, c->p.cutoff, c->st);
    c->n_launches += 1;
    TKHP_CUDA(c, cudaGetLastError());
    return TKHP_OK;
}

// first block of every group: fixed for the life of the context (tkhp_create, which synchronises)
int cluster_init(Ctx *c) {
    if (c->p.list_mode == TKHP_LIST_TILES) return TKHP_OK;
    ClusterWs ws = get_ws(c);
    k_group_first<<<div_up(ws.n_groups + 1, 256), 256>>>(ws.group_first, ws.n_groups, c->n_blocks);
    TKHP_CUDA(c, cudaGetLastError());
    return TKHP_OK;
}

long long cluster_slots(Ctx *c) { return 8LL * c->h_state->n_cluster_entries; }

}  // namespace tkhp
