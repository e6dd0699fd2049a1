// atom_stored.cu -- ATOM list mode with STORED real-space matrix elements (SURVEY 8(f) NEXT #1b).
//
// Paper, "OpenACC optimisations", polarization solver: "precompute the real space matrix elements
// before the iterations".  For the positions of a list build the two radial factors of
// every listed pair, G1 = bn1 - (1 - lambda3)/R^3 and G2/3 = [bn2 - 3 (1 - lambda5)/R^5]/3 (DESIGN.md
// section 2, T1-T2), do not change from one T.mu product to the next: k_atom_tstore evaluates them
// once (same FAR/NEAR formulas as the pair kernel, FP32) and writes one float2 per list slot, in the
// layout of the lists themselves ([block][row][lane][8 entries], 64 bytes per lane and row), and
// k_atom_tmu_stored applies them: per pair 24 bytes of shared memory (the staged record), 8 bytes of
// the stored stream and 13 FMA-pipe cycles instead of 28 (FAR) / 40 (NEAR).  The price is the stream:
// 8 bytes per slot and product from HBM/L2 (config 2: 119 MB per product, the 126 MB L2 keeps part of
// it between the products of a solve), so this product is bound by HBM bandwidth, not by the FMA pipe.
//
// Selected by tkhp_params.solver_flags & TKHP_SOLVER_STORED_T (MIXED / FIXED precision, ATOM lists):
// tkhp_tmatvec and the launch-per-matvec PCG path then use the stored product; the elements are
// computed lazily by the first product after a list build and stay valid until the next build.
#include "atom_tmu.cuh"
#include "atom_epilogue.cuh"

namespace tkhp {

// ---- the two radial factors of one pair, scalar FP32 (the formulas of tmu_far2 / tmu_near2)
__device__ __forceinline__ float2 radial_far(float s, const TmuConsts &K) {
    const float t = fast_rsqrt(s);
    const float ez = fast_ex2(s * K.nb2l);
    const float t2 = t * t;
    float q = fmaf(K.q[5], t, K.q[4]);
    q = fmaf(q, t, K.q[3]);
    q = fmaf(q, t, K.q[2]);
    q = fmaf(q, t, K.q[1]);
    q = fmaf(q, t, K.q[0]);
    const float aq = fmaf(t2, q, K.c1b);
    const float G1 = (ez * t2) * aq;
    const float G2 = t2 * fmaf(K.k3, ez, G1);                      // G2 / 3
    return make_float2(G1, G2);
}
__device__ __forceinline__ float2 radial_near(float s, float wlw, const TmuConsts &K) {
    constexpr float c[TKHP_ERFCX_DEG + 1] = TKHP_ERFCX_COEFFS;
    constexpr float LN2 = 0.69314718055994531f;
    const float rinv = fast_rsqrt(s);
    const float r = s * rinv;
    const float u = fast_rcp(fmaf(r, K.pb, 1.0f));
    const float ez = fast_ex2(s * K.nb2l);
    const float r3 = s * r;
    const float xl = r3 * wlw;                                     // x log2 e
    const float et = fast_ex2(-xl);
    float p = c[TKHP_ERFCX_DEG];
#pragma unroll
    for (int d = TKHP_ERFCX_DEG - 1; d >= 0; --d) p = fmaf(p, u, c[d]);
    const float g1 = fmaf(r, K.c1b, p);                            // erfcx(z) + c z
    const float a1 = fmaf(ez, g1, -et);                            // R^3 G1
    const float h2 = fmaf(r3, K.k3, g1);
    const float x = xl * LN2;
    const float xe = fmaf(x, et, et);                              // (1 + x) e^-x
    const float b2 = fmaf(ez, h2, -xe);                            // R^5 G2 / 3
    const float rinv2 = rinv * rinv, rinv3 = rinv2 * rinv;
    return make_float2(a1 * rinv3, b2 * (rinv2 * rinv3));
}

// one row of 8 entries: the factors of each entry
template <bool FARF>
__device__ __forceinline__ void store_row(const TmuSmem &S, const uint4 &e, const TmuLane &L, const TmuConsts &K,
                                          uint4 *__restrict__ out) {
    const unsigned wd[4] = {e.x, e.y, e.z, e.w};
    float2 g[8];
#pragma unroll
    for (int h = 0; h < 8; ++h) {
        const unsigned off = (wd[h >> 1] >> ((h & 1) * 16)) & 0xffffu;
        const float4 p = *reinterpret_cast<const float4 *>(S.a + off);
        const float Dx = p.x - lo(L.pxy), Dy = p.y - hi(L.pxy), Dz = p.z + L.nz;
        const float s = fmaf(Dz, Dz, fmaf(Dy, Dy, Dx * Dx));
        if (FARF) {
            g[h] = radial_far(s, K);
        } else {
            const float w = *reinterpret_cast<const float *>(S.w + (off >> 2));
            g[h] = radial_near(s, w * L.wl, K);
        }
    }
#pragma unroll
    for (int q = 0; q < 4; ++q)
        out[q] = make_uint4(__float_as_uint(g[2 * q].x), __float_as_uint(g[2 * q].y), __float_as_uint(g[2 * q + 1].x),
                            __float_as_uint(g[2 * q + 1].y));
}

// ---- precompute: one CTA per group, one warp per block (staging as in k_atom_tmu32, positions only)
template <bool FAR>
__global__ void __launch_bounds__(GT, 2)
k_atom_tstore(ClusterWs ws, const float4 *__restrict__ gpos, const float4 *__restrict__ stage_pos, TmuConsts K,
              uint4 *__restrict__ tstore, int s_chunk) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int pstride = s_chunk + N_DUMMY;
    float4 *s_a = reinterpret_cast<float4 *>(smem_raw);
    float *s_w = reinterpret_cast<float *>(smem_raw + (size_t)24 * pstride);
    TmuSmem S;
    S.a = smem_raw; S.b = smem_raw + (size_t)16 * pstride; S.w = smem_raw + (size_t)24 * pstride;
    const int g = blockIdx.x, t = threadIdx.x, lane = t & 31, w = t >> 5;
    const int b0 = ws.group_first[g], nb = ws.group_first[g + 1] - b0;
    const int count = ws.stage_count[g];
    const int n_chunks = atom_chunks_of(count, s_chunk);
    const size_t gbase = (size_t)g * ws.s_cap;
    const bool active = w < nb && n_chunks <= NCH_MAX;
    const int blk = b0 + (w < nb ? w : 0);
    const int2 *__restrict__ seg = ws.aseg + (size_t)blk * NSEG_MAX;
    const int rows_cap = ws.a_cap >> 3;
    const uint4 *__restrict__ rows = reinterpret_cast<const uint4 *>(ws.alist + (size_t)blk * ws.a_cap * 32) + lane;
    uint4 *__restrict__ out = tstore + ((size_t)blk * rows_cap * 32 + lane) * 4;      // row r of this lane: out[r * 128 .. + 4]
    TmuLane L;
    {
        const float4 pi = gpos[blk * BLOCK + lane];
        L.pxy = pk(pi.x, pi.y);
        L.nz = -pi.z;
        L.wl = pi.w * 1.4426950408889634f;
    }
    if (t < N_DUMMY) {
        const float far = -2.0f * PHANTOM_FAR;
        const int dmy = atom_dummy_index(count, n_chunks) + t;
        s_a[dmy] = make_float4(far, far, far, 0.f);
        s_w[dmy] = 0.f;
    }
    int d = 0;
    int2 sd = seg[0];
    for (int c = 0; c < n_chunks; ++c) {
        __syncthreads();
        for (int l = t, idx = c + t * n_chunks; idx < count; l += GT, idx += GT * n_chunks) {
            const float4 p = stage_pos[gbase + idx];
            s_a[l] = make_float4(p.x, p.y, p.z, 0.f);
            s_w[l] = p.w;
        }
        __syncthreads();
        if (!active) continue;
        while (seg_chunk(sd) == c) {
            const int row0 = seg_row0(sd);
            const int fr = (seg_far_calls(sd) + 3) >> 2, nr = (seg_near_calls(sd) + 3) >> 2;
            for (int r = row0; r < row0 + fr; ++r) store_row<FAR>(S, ldg_row(rows + (size_t)r * 32), L, K, out + (size_t)r * 128);
            for (int r = row0 + fr; r < row0 + fr + nr; ++r) store_row<false>(S, ldg_row(rows + (size_t)r * 32), L, K, out + (size_t)r * 128);
            sd = seg[++d];
        }
    }
}

// ---- the product with stored factors: two entries of one lane
__device__ __forceinline__ void tmu_stored2(const TmuSmem &S, unsigned off0, unsigned off1, const uint4 &g, const TmuLane &L,
                                            PartialTmu &A) {
    const ulonglong2 p0 = *reinterpret_cast<const ulonglong2 *>(S.a + off0);          // (x,y) (z,mu_z)
    const ulonglong2 p1 = *reinterpret_cast<const ulonglong2 *>(S.a + off1);
    const f2 m0 = *reinterpret_cast<const f2 *>(S.b + (off0 >> 1));                   // (mu_x, mu_y)
    const f2 m1 = *reinterpret_cast<const f2 *>(S.b + (off1 >> 1));
    const f2 Dxy0 = sub2(p0.x, L.pxy), Dxy1 = sub2(p1.x, L.pxy);
    const float Dz0 = lo(p0.y) + L.nz, Dz1 = lo(p1.y) + L.nz;
    float d0 = lo(m0) * lo(Dxy0), d1 = lo(m1) * lo(Dxy1);
    d0 = fmaf(hi(m0), hi(Dxy0), d0); d1 = fmaf(hi(m1), hi(Dxy1), d1);
    d0 = fmaf(hi(p0.y), Dz0, d0); d1 = fmaf(hi(p1.y), Dz1, d1);
    const float G10 = __uint_as_float(g.x), G20 = __uint_as_float(g.y), G11 = __uint_as_float(g.z), G21 = __uint_as_float(g.w);
    const float c0 = G20 * d0, c1 = G21 * d1;
    A.cxy = fma2(Dxy0, bc(c0), A.cxy); A.cz = fmaf(c0, Dz0, A.cz);
    A.mxy = fma2(m0, bc(G10), A.mxy); A.mz = fmaf(G10, hi(p0.y), A.mz);
    A.cxy = fma2(Dxy1, bc(c1), A.cxy); A.cz = fmaf(c1, Dz1, A.cz);
    A.mxy = fma2(m1, bc(G11), A.mxy); A.mz = fmaf(G11, hi(p1.y), A.mz);
}

__device__ __forceinline__ uint4 ldg_stream(const uint4 *p) {
    uint4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    return v;
}

// One CTA per group, one warp per block; a group with few blocks gives every block to 2, 4 or 8
// warps (rows part, part + wpb, ...).  A row (entries 16 B + factors 64 B per lane) is loaded one row
// before its use.
__global__ void __launch_bounds__(GT, 3)
k_atom_tmu_stored(ClusterWs ws, const float4 *__restrict__ stage_pos, const float4 *__restrict__ mu,
                  const uint4 *__restrict__ tstore, double *__restrict__ acc, int n_pad, int s_chunk, int fixed,
                  DeviceState *st, int iter, PcgFuse fuse) {
    if (iter >= 0 && iter >= st->conv_at) return;      // PCG already converged (pcg.cu)
    constexpr int SU = 4;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int pstride = s_chunk + N_DUMMY;
    float4 *s_a = reinterpret_cast<float4 *>(smem_raw);
    float2 *s_b = reinterpret_cast<float2 *>(smem_raw + (size_t)16 * pstride);
    TmuSmem S;
    S.a = smem_raw; S.b = smem_raw + (size_t)16 * pstride; S.w = smem_raw + (size_t)24 * pstride;
    const int g = blockIdx.x, t = threadIdx.x, lane = t & 31, w = t >> 5;
    const int b0 = ws.group_first[g], nb = ws.group_first[g + 1] - b0;
    const int count = ws.stage_count[g];
    const int n_chunks = atom_chunks_of(count, s_chunk);
    const size_t gbase = (size_t)g * ws.s_cap;
    const int wpb = warps_per_block(nb);
    const int kb = w / wpb, part = w - kb * wpb;
    const bool active = kb < nb && n_chunks <= NCH_MAX;
    const int blk = b0 + (kb < nb ? kb : 0);
    const int slot = blk * BLOCK + lane;
    const int2 *__restrict__ seg = ws.aseg + (size_t)blk * NSEG_MAX;
    const int rows_cap = ws.a_cap >> 3;
    const uint4 *__restrict__ rows = reinterpret_cast<const uint4 *>(ws.alist + (size_t)blk * ws.a_cap * 32) + lane;
    const uint4 *__restrict__ fac = tstore + ((size_t)blk * rows_cap * 32 + lane) * 4;
    TmuLane L;
    {
        const float4 pi = ws.gpos32[slot];
        L.pxy = pk(pi.x, pi.y);
        L.nz = -pi.z;
        L.wl = 0.f;
    }
    double dx = 0.0, dy = 0.0, dz = 0.0;
    PartialTmu A;
    if (t < N_DUMMY) {
        const float far = -2.0f * PHANTOM_FAR;
        const int dmy = atom_dummy_index(count, n_chunks) + t;
        s_a[dmy] = make_float4(far, far, far, 0.f);
        s_b[dmy] = make_float2(0.f, 0.f);
    }
    int d = 0, n_rows = 0;
    int2 sd = seg[0];
    int tg = part;                                   // my next row
    // row tg of this lane: entries and factors, one row ahead (clamped: the list area of a block has >= 8 rows)
    const int last = rows_cap - 1;
    uint4 e_n = ldg_row(rows + (size_t)min(tg, last) * 32);
    uint4 f_n[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) f_n[q] = ldg_stream(fac + (size_t)min(tg, last) * 128 + q);
    for (int c = 0; c < n_chunks; ++c) {
        __syncthreads();
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
                }
            }
        }
        __syncthreads();
        if (!active) continue;
        while (seg_chunk(sd) == c) {
            const int rend = seg_row0(sd) + ((seg_far_calls(sd) + 3) >> 2) + ((seg_near_calls(sd) + 3) >> 2);
            for (; tg < rend; tg += wpb) {
                const uint4 e = e_n;
                uint4 f[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) f[q] = f_n[q];
                const int nx = min(tg + wpb, last);
                e_n = ldg_row(rows + (size_t)nx * 32);
#pragma unroll
                for (int q = 0; q < 4; ++q) f_n[q] = ldg_stream(fac + (size_t)nx * 128 + q);
                const unsigned wd[4] = {e.x, e.y, e.z, e.w};
#pragma unroll
                for (int q = 0; q < 4; ++q) tmu_stored2(S, wd[q] & 0xffffu, wd[q] >> 16, f[q], L, A);
                if ((++n_rows & 3) == 0) A.flush(dx, dy, dz, fixed);
            }
            sd = seg[++d];
        }
    }
    A.flush(dx, dy, dz, fixed);
    dx = acc_value(dx, fixed != 0); dy = acc_value(dy, fixed != 0); dz = acc_value(dz, fixed != 0);
    pair_epilogue<true>(smem_raw, dx, dy, dz, wpb, part, kb < nb, slot, n_pad, acc, st, fuse);
}

// ----------------------------------------------------------------------------- host side
size_t atom_stored_bytes(const tkhp_params *p, int n_blocks) {
    if (!(p->solver_flags & TKHP_SOLVER_STORED_T) || p->list_mode != TKHP_LIST_ATOM || p->precision == TKHP_FP64) return 0;
    ClusterWs ws;
    carve_cluster(p, n_blocks, nullptr, &ws);
    return (size_t)n_blocks * (size_t)ws.a_cap * 32 * sizeof(float2);
}

int atom_stored_configure(Ctx *c) {
    const int big = (int)tmu32_smem(atom_chunk_capacity(false, 0));
    TKHP_CUDA(c, cudaFuncSetAttribute(k_atom_tstore<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, big));
    TKHP_CUDA(c, cudaFuncSetAttribute(k_atom_tstore<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, big));
    TKHP_CUDA(c, cudaFuncSetAttribute(k_atom_tmu_stored, cudaFuncAttributeMaxDynamicSharedMemorySize, big));
    return TKHP_OK;
}

static TmuConsts stored_consts(Ctx *c) {
    const double b = c->p.ewald_beta;
    TmuConsts K;
    K.pb = (float)((double)TKHP_ERFCX_P * b);
    K.nb2l = (float)(-1.4426950408889634 * b * b);
    K.c1b = (float)(2.0 / SQRT_PI * b);
    K.k3 = (float)(4.0 / (3.0 * SQRT_PI) * b * b * b);
    for (int k = 0; k < 6; ++k) K.q[k] = c->far_q[k];
    K.fixed = c->fixed ? 1 : 0;
    return K;
}

// acc = T_real * mu32 with the stored factors (computed first if the list is newer than they are)
int atom_stored_tmatvec(Ctx *c, cudaStream_t s) {
    ClusterWs ws = get_ws(c);
    const int s_chunk = atom_chunk_capacity(false, ws.chunk_cap);
    const size_t smem = tmu32_smem(s_chunk);
    if (!c->tstore_valid) {
        const TmuConsts K = stored_consts(c);
        if (c->far_on)
            k_atom_tstore<true><<<ws.n_groups, GT, smem, s>>>(ws, ws.gpos32, ws.stage_pos32, K, c->tstore, s_chunk);
        else
            k_atom_tstore<false><<<ws.n_groups, GT, smem, s>>>(ws, ws.gpos32, ws.stage_pos32, K, c->tstore, s_chunk);
        c->n_launches += 1;
        c->tstore_valid = true;
    }
    PcgFuse fuse;
    fuse.on = c->fuse_q;
    const double b = c->p.ewald_beta;
    fuse.self = 4.0 * b * b * b / (3.0 * SQRT_PI);
    fuse.vp = c->vp; fuse.inv_alpha = c->inv_alpha_s; fuse.vq = c->vq;
    fuse.part = c->partials + 2 * (size_t)c->part_cap;
    k_atom_tmu_stored<<<ws.n_groups, GT, smem, s>>>(ws, ws.stage_pos32, c->mu32, c->tstore, c->acc, c->n_pad, s_chunk,
                                                     c->fixed ? 1 : 0, c->st, c->spec_iter, fuse);
    c->n_launches += 1;
    TKHP_CUDA(c, cudaGetLastError());
    return TKHP_OK;
}

}  // namespace tkhp
