// atom_tmu.cuh -- the packed-FP32 T.mu pair arithmetic of the ATOM list mode, shared by the
// stand-alone pair kernel (atom_pairs.cu) and the persistent PCG kernel (atom_solve.cu).
// DESIGN.md section 5.3; formulas: DESIGN.md section 2 (T1, T2).
#pragma once
#include "cluster.cuh"
#include "f32x2.cuh"

namespace tkhp {

// ---- FP32 partial sums of one lane ------------------------------------------------------------
// Two partials, C = sum G2/3 (mu_j.D) D and M = sum G1 mu_j (D = r_j - r_i), so that the pair loop
// needs neither the factor 3 nor a negation; (T mu)_i = 3 C - M is formed at every flush into the
// FP64 registers.
struct PartialTmu {
    f2 cxy = 0ull, mxy = 0ull;
    float cz = 0.f, mz = 0.f;
    // into the 64-bit containers: FP64, or int64 fixed point (TKHP_FIXED, common.cuh acc_add)
    __device__ __forceinline__ void flush(double &dx, double &dy, double &dz, int fixed) {
        acc_add(dx, fmaf(3.0f, lo(cxy), -lo(mxy)), fixed != 0);
        acc_add(dy, fmaf(3.0f, hi(cxy), -hi(mxy)), fixed != 0);
        acc_add(dz, fmaf(3.0f, cz, -mz), fixed != 0);
        cxy = 0ull; mxy = 0ull; cz = 0.f; mz = 0.f;
    }
};

// ---- packed FP32 T.mu: two list entries of one lane per call ------------------------------------
// Staged records: A[idx] = (x, y, z, mu_z) (16 B), B[idx] = (mu_x, mu_y) (8 B), W[idx] = w (4 B); an
// entry is the byte offset of A[idx].  The two pairs (j0, j1) of a lane share every instruction of
// the radial chain (lo half = j0, hi half = j1); the geometry and the 3-vector updates are packed
// over (x, y), the register pairs the loads deliver them in.
struct TmuLane {
    f2 pxy;         // (x_i, y_i)
    float nz;       // -z_i
    float wl;       // w_i log2 e
};
struct TmuConsts {
    float pb;       // P beta (TKHP_ERFCX_P): u = 1 / (1 + pb R)
    float nb2l;     // -beta^2 log2 e:        e^{-z^2} = ex2(nb2l R^2)
    float c1b;      // (2/sqrt pi) beta:      c z = c1b R
    float k3;       // (4/(3 sqrt pi)) beta^3: (2c/3) z^3 = k3 R^3
    float q[6];     // far fit: erfcx(beta R) = t (q0 + q1 t + ... + q5 t^5), t = 1/R
    int fixed;      // TKHP_FIXED: the 64-bit accumulators are int64 with 34 fractional bits
};
struct TmuSmem {
    const unsigned char *a, *b, *w;   // generic pointers into shared memory
};

// FAR pair: with t = 1/R, t2 = t^2, ez = e^{-z^2}, Q(t) the fit above,
//   G1   = bn1 = ez t2 (t2 Q + c1b),        G2/3 = bn2/3 = t2 (G1 + k3 ez).
// Per pair: 2 MUFU (rsqrt, ex2) and 12 packed + 16 scalar FMA-pipe operations.
__device__ __forceinline__ void tmu_far2(const TmuSmem &S, unsigned off0, unsigned off1, const TmuLane &L,
                                         const TmuConsts &K, PartialTmu &A) {
    const ulonglong2 p0 = *reinterpret_cast<const ulonglong2 *>(S.a + off0);          // (x,y) (z,mu_z)
    const ulonglong2 p1 = *reinterpret_cast<const ulonglong2 *>(S.a + off1);
    const f2 m0 = *reinterpret_cast<const f2 *>(S.b + (off0 >> 1));                   // (mu_x, mu_y)
    const f2 m1 = *reinterpret_cast<const f2 *>(S.b + (off1 >> 1));
    const f2 Dxy0 = sub2(p0.x, L.pxy), Dxy1 = sub2(p1.x, L.pxy);
    const float Dz0 = lo(p0.y) + L.nz, Dz1 = lo(p1.y) + L.nz;
    float s0 = lo(Dxy0) * lo(Dxy0), s1 = lo(Dxy1) * lo(Dxy1);
    s0 = fmaf(hi(Dxy0), hi(Dxy0), s0); s1 = fmaf(hi(Dxy1), hi(Dxy1), s1);
    s0 = fmaf(Dz0, Dz0, s0); s1 = fmaf(Dz1, Dz1, s1);
    const f2 r2 = pk(s0, s1);
    const f2 t = pk(fast_rsqrt(s0), fast_rsqrt(s1));
    const f2 ea = mul2(r2, bc(K.nb2l));
    const f2 ez = pk(fast_ex2(lo(ea)), fast_ex2(hi(ea)));
    const f2 t2 = mul2(t, t);
    f2 q = fma2(bc(K.q[5]), t, bc(K.q[4]));
    q = fma2(q, t, bc(K.q[3]));
    q = fma2(q, t, bc(K.q[2]));
    q = fma2(q, t, bc(K.q[1]));
    q = fma2(q, t, bc(K.q[0]));
    const f2 aq = fma2(t2, q, bc(K.c1b));
    const f2 e2 = mul2(ez, t2);
    const f2 G1 = mul2(e2, aq);
    const f2 G2 = mul2(t2, fma2(bc(K.k3), ez, G1));                    // G2 / 3
    float d0 = lo(m0) * lo(Dxy0), d1 = lo(m1) * lo(Dxy1);
    d0 = fmaf(hi(m0), hi(Dxy0), d0); d1 = fmaf(hi(m1), hi(Dxy1), d1);
    d0 = fmaf(hi(p0.y), Dz0, d0); d1 = fmaf(hi(p1.y), Dz1, d1);
    const f2 cc = mul2(G2, pk(d0, d1));
    A.cxy = fma2(Dxy0, bc(lo(cc)), A.cxy); A.cz = fmaf(lo(cc), Dz0, A.cz);
    A.mxy = fma2(m0, bc(lo(G1)), A.mxy); A.mz = fmaf(lo(G1), hi(p0.y), A.mz);
    A.cxy = fma2(Dxy1, bc(hi(cc)), A.cxy); A.cz = fmaf(hi(cc), Dz1, A.cz);
    A.mxy = fma2(m1, bc(hi(G1)), A.mxy); A.mz = fmaf(hi(G1), hi(p1.y), A.mz);
}

// NEAR pair: the full formula (pair_math.cuh), erfcx by the degree-7 polynomial in u = 1/(1 + pb R).
// Per pair: 4 MUFU (rsqrt, rcp, 2 ex2) and 41 FMA-pipe cycles.
__device__ __forceinline__ void tmu_near2(const TmuSmem &S, unsigned off0, unsigned off1, const TmuLane &L,
                                          const TmuConsts &K, PartialTmu &A) {
    constexpr float c[TKHP_ERFCX_DEG + 1] = TKHP_ERFCX_COEFFS;
    constexpr float LN2 = 0.69314718055994531f;
    const ulonglong2 p0 = *reinterpret_cast<const ulonglong2 *>(S.a + off0);
    const ulonglong2 p1 = *reinterpret_cast<const ulonglong2 *>(S.a + off1);
    const f2 m0 = *reinterpret_cast<const f2 *>(S.b + (off0 >> 1));
    const f2 m1 = *reinterpret_cast<const f2 *>(S.b + (off1 >> 1));
    const float w0 = *reinterpret_cast<const float *>(S.w + (off0 >> 2));
    const float w1 = *reinterpret_cast<const float *>(S.w + (off1 >> 2));
    const f2 Dxy0 = sub2(p0.x, L.pxy), Dxy1 = sub2(p1.x, L.pxy);
    const float Dz0 = lo(p0.y) + L.nz, Dz1 = lo(p1.y) + L.nz;
    float s0 = lo(Dxy0) * lo(Dxy0), s1 = lo(Dxy1) * lo(Dxy1);
    s0 = fmaf(hi(Dxy0), hi(Dxy0), s0); s1 = fmaf(hi(Dxy1), hi(Dxy1), s1);
    s0 = fmaf(Dz0, Dz0, s0); s1 = fmaf(Dz1, Dz1, s1);
    const f2 r2 = pk(s0, s1);
    const f2 rinv = pk(fast_rsqrt(s0), fast_rsqrt(s1));
    const f2 r = mul2(r2, rinv);
    const f2 ua = fma2(r, bc(K.pb), bc(1.0f));
    const f2 u = pk(fast_rcp(lo(ua)), fast_rcp(hi(ua)));
    const f2 ea = mul2(r2, bc(K.nb2l));
    const f2 ez = pk(fast_ex2(lo(ea)), fast_ex2(hi(ea)));
    const f2 r3 = mul2(r2, r);
    const f2 xl = mul2(r3, pk(w0 * L.wl, w1 * L.wl));                // x log2 e
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
    float d0 = lo(m0) * lo(Dxy0), d1 = lo(m1) * lo(Dxy1);
    d0 = fmaf(hi(m0), hi(Dxy0), d0); d1 = fmaf(hi(m1), hi(Dxy1), d1);
    d0 = fmaf(hi(p0.y), Dz0, d0); d1 = fmaf(hi(p1.y), Dz1, d1);
    const f2 cc = mul2(G2, pk(d0, d1));
    A.cxy = fma2(Dxy0, bc(lo(cc)), A.cxy); A.cz = fmaf(lo(cc), Dz0, A.cz);
    A.mxy = fma2(m0, bc(lo(G1)), A.mxy); A.mz = fmaf(lo(G1), hi(p0.y), A.mz);
    A.cxy = fma2(Dxy1, bc(hi(cc)), A.cxy); A.cz = fmaf(hi(cc), Dz1, A.cz);
    A.mxy = fma2(m1, bc(hi(G1)), A.mxy); A.mz = fmaf(hi(G1), hi(p1.y), A.mz);
}

constexpr int TMU_REC = 28;          // staged bytes per record: A 16 + B 8 + W 4

__host__ __device__ inline size_t tmu32_smem(int s_chunk) { return ((size_t)TMU_REC * (s_chunk + N_DUMMY) + 15) & ~(size_t)15; }

// One row (8 entries per lane) of FAR or NEAR pairs; n < 4: the last row of a class.
template <bool FARF>
__device__ __forceinline__ void tmu_row(const TmuSmem &S, const uint4 &e, int n, const TmuLane &L, const TmuConsts &K,
                                        PartialTmu &A) {
    if (n >= 4) {                              // straight-line: four independent chains interleave
        const unsigned wd[4] = {e.x, e.y, e.z, e.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (FARF) tmu_far2(S, wd[k] & 0xffffu, wd[k] >> 16, L, K, A);
            else tmu_near2(S, wd[k] & 0xffffu, wd[k] >> 16, L, K, A);
        }
    } else {
        for (int k = 0; k < n; ++k) {
            const unsigned x = k == 0 ? e.x : (k == 1 ? e.y : e.z);
            if (FARF) tmu_far2(S, x & 0xffffu, x >> 16, L, K, A);
            else tmu_near2(S, x & 0xffffu, x >> 16, L, K, A);
        }
    }
}

// one lane's row of list entries (16 bytes), read-only path, pinned in program order
__device__ __forceinline__ uint4 ldg_row(const uint4 *p) {
    uint4 v;
    asm volatile("ld.global.nc.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    return v;
}
// warps per block: a group with few blocks (small systems: config 1 has 1.7 blocks per group) gives
// each block to 2, 4 or 8 warps; warp `part` of a block takes the block's list rows part,
// part + wpb, ... and the parts are added in a fixed order at the end (bit-reproducible)
__device__ __forceinline__ int warps_per_block(int nb) { return nb >= 5 ? 1 : (nb >= 3 ? 2 : (nb == 2 ? 4 : 8)); }

// A warp's stream of list rows: my rows are part, part + wpb, ... of the block's rows, whatever
// segment they fall in.  A row (16 bytes per lane) is loaded into registers two rows before its use.
struct RowStream {
    const uint4 *rp;
    int n_load, step;
    uint4 e1, e2;
    __device__ __forceinline__ void open(const uint4 *rows_of_lane, int t_total, int part, int wpb) {
        n_load = t_total > part ? (t_total - part + wpb - 1) / wpb : 0;       // my rows not yet requested
        rp = rows_of_lane + (size_t)part * 32;
        step = 32 * wpb;
        e1 = make_uint4(0, 0, 0, 0);
        e2 = e1;
        if (n_load > 0) { e1 = ldg_row(rp); rp += step; --n_load; }
        if (n_load > 0) { e2 = ldg_row(rp); rp += step; --n_load; }
    }
    __device__ __forceinline__ uint4 next() {
        const uint4 e = e1;
        e1 = e2;
        if (n_load > 0) { e2 = ldg_row(rp); rp += step; --n_load; }
        return e;
    }
};

// All segments of chunk c of one block: FAR rows, then NEAR rows, of every segment.  `tg` is my next
// row, (sd, d) the descriptor cursor; FP32 partials go to the FP64 registers every 4 rows.
template <bool FAR>
__device__ __forceinline__ void tmu_walk(const int2 *__restrict__ seg, int c, int &d, int2 &sd, int &tg, int wpb,
                                         RowStream &R, const TmuSmem &S, const TmuLane &L, const TmuConsts &K,
                                         PartialTmu &A, int &n_rows, double &dx, double &dy, double &dz) {
    while (seg_chunk(sd) == c) {
        const int row0 = seg_row0(sd);
        const int ncf = seg_far_calls(sd), ncn = seg_near_calls(sd);
        // first class of rows (FAR pairs, or every pair when the far class is off)
        const int f_full = row0 + (ncf >> 2);
        for (; tg < f_full; tg += wpb) {
            const uint4 e = R.next();
            tmu_row<FAR>(S, e, 4, L, K, A);
            if ((++n_rows & 3) == 0) A.flush(dx, dy, dz, K.fixed);   // every 32 entries: FP32 partial -> 64-bit container
        }
        if ((ncf & 3) && tg == f_full) {
            const uint4 e = R.next();
            tmu_row<FAR>(S, e, ncf & 3, L, K, A);
            tg += wpb;
        }
        const int n0 = row0 + ((ncf + 3) >> 2), n_full = n0 + (ncn >> 2);
        for (; tg < n_full; tg += wpb) {
            const uint4 e = R.next();
            tmu_row<false>(S, e, 4, L, K, A);
            if ((++n_rows & 3) == 0) A.flush(dx, dy, dz, K.fixed);
        }
        if ((ncn & 3) && tg == n_full) {
            const uint4 e = R.next();
            tmu_row<false>(S, e, ncn & 3, L, K, A);
            tg += wpb;
        }
        sd = seg[++d];
    }
}

}  // namespace tkhp
