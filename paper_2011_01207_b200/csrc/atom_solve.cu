// atom_solve.cu -- the whole PCG solve as ONE persistent cooperative kernel (MIXED precision, ATOM lists).
//
// Paper: "(polarization) matrix-vector product at each iteration" of a "preconditioned conjugate
// gradient" with "a diagonal preconditioner"; the solver is host-driven there
// (OpenACC kernels per vector operation).  Recurrences: DESIGN.md section 2 "S".
//
// B200 design.  With one launch per matvec, every iteration re-stages the
// group's neighbourhood (positions that never change during a solve), pays two kernel launches and
// drains the SMs in between: 13 of 43 us per matvec on config 2.  Here one CTA per group stays
// resident for the whole solve:
//  * the staged positions, Thole factors and staging indices are loaded ONCE; per iteration only
//    the operand vector is gathered (16 bytes per staged atom);
//  * every lane owns one atom for the whole solve: its mu, r and p live in shared memory (FP64), q
//    in registers; the vector updates of an iteration are done by the owner, between two grid
//    barriers;
//  * dot products: one FP64 partial per CTA, then EVERY CTA adds all partials in the same order,
//    so all CTAs hold identical totals and take the same convergence decision (deterministic, no
//    floating-point atomics, bit-reproducible);
//  * the direction p is carried in FP32 by everybody who needs it: the owner publishes
//    u = fp32(alpha r) BEFORE the barrier that completes r.z, and each CTA forms
//    p_j <- u_j + delta p_j for its staged atoms (and the owner for its own atom) with the same FP32
//    arithmetic afterwards.  The operand of T and the p of the vector updates are then the SAME
//    numbers, and an iteration needs two grid barriers instead of three;
//  * a grid barrier is one atomic per CTA on a monotonic counter and a spin on a release word.
// Requirements (else do_polar_solve keeps the launch-per-matvec path): every group's neighbourhood
// fits one chunk, and the grid is co-resident (cooperative launch).
#include "atom_tmu.cuh"
#include "reduce.cuh"

namespace tkhp {

struct SolveArgs {
    ClusterWs ws;
    const float4 *gpos;        // n_pad: own atoms, group frame
    const float4 *stage_pos;   // n_groups * s_cap
    float4 *mu0;               // n_pad: the initial guess, packed by the owners (sorted order)
    float4 *u32;               // n_pad: u = fp32(alpha r), published by the owners before the barrier that completes r.z
    TmuConsts K;
    const double *field;       // N x 3, caller's order
    double *mu;                // N x 3, caller's order: in (guess) / out
    const int32_t *perm;       // n_pad: sorted slot -> caller's atom, -1 = phantom
    int use_guess;
    volatile double *result;   // host-mapped: |r|^2, iterations, barrier time-out flag
    const double *alpha_s, *inv_alpha_s;
    double *part_a, *part_b;   // 2 * n_groups each
    DeviceState *st;
    double tol, self;
    int max_iter, n_atoms, n_pad, s_chunk, rot_div;
    int test_fault;          // TKHP_SOLVER_TEST_BARRIER_FAULT: the last CTA never arrives at the first barrier
};

__host__ __device__ inline size_t solve_smem(int s_chunk, bool split) {
    size_t b = ((size_t)TMU_REC * (s_chunk + N_DUMMY) + 15) & ~(size_t)15;   // A, B, W
    b += (size_t)4 * s_chunk;                                         // staging indices
    b = (b + 15) & ~(size_t)15;
    if (split) b += (size_t)GB * 96 * sizeof(double);                 // parts of a shared block
    b += (size_t)6 * GT * sizeof(double);                             // mu, r of the owners
    b += (size_t)3 * GT * sizeof(float);                              // p of the owners (FP32)
    return b;
}

template <bool FAR, bool SPLIT>
__global__ void __launch_bounds__(GT, 3)
k_pcg_persist(SolveArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int s_chunk = a.s_chunk, pstride = s_chunk + N_DUMMY;
    float4 *s_a = reinterpret_cast<float4 *>(smem_raw);
    float2 *s_b = reinterpret_cast<float2 *>(smem_raw + (size_t)16 * pstride);
    float *s_w = reinterpret_cast<float *>(smem_raw + (size_t)24 * pstride);
    size_t off = ((size_t)TMU_REC * pstride + 15) & ~(size_t)15;
    int *s_idx = reinterpret_cast<int *>(smem_raw + off);
    off = (off + (size_t)4 * s_chunk + 15) & ~(size_t)15;
    double *s_part = reinterpret_cast<double *>(smem_raw + off);
    if (SPLIT) off += (size_t)GB * 96 * sizeof(double);
    double *s_vec = reinterpret_cast<double *>(smem_raw + off);      // [6][GT]: mu xyz, r xyz
    off += (size_t)6 * GT * sizeof(double);
    float *s_p = reinterpret_cast<float *>(smem_raw + off);          // [3][GT]
    TmuSmem S;
    S.a = smem_raw; S.b = smem_raw + (size_t)16 * pstride; S.w = smem_raw + (size_t)24 * pstride;

    const ClusterWs &ws = a.ws;
    const int g = blockIdx.x, t = threadIdx.x, lane = t & 31, w = t >> 5;
    const int b0 = ws.group_first[g], nb = ws.group_first[g + 1] - b0;
    const int count = ws.stage_count[g];
    const size_t gbase = (size_t)g * ws.s_cap;
    const int wpb = SPLIT ? warps_per_block(nb) : 1;
    const int kb = SPLIT ? w / wpb : ((w + g / a.rot_div) & (GB - 1)), part = SPLIT ? w - kb * wpb : 0;
    const bool active = kb < nb;
    const bool owner = active && part == 0;
    const int blk = b0 + (active ? kb : 0);
    const int slot = blk * BLOCK + lane;
    const int n_pad = a.n_pad;
    const int2 *__restrict__ seg = ws.aseg + (size_t)blk * NSEG_MAX;
    const uint4 *rows = reinterpret_cast<const uint4 *>(ws.alist + (size_t)blk * ws.a_cap * 32) + lane;
    const int t_total = active ? seg_row0(seg[NSEG_MAX - 1]) : 0;
    DeviceState *st = a.st;

    TmuLane L;
    {
        const float4 pi = a.gpos[slot];
        L.pxy = pk(pi.x, pi.y);
        L.nz = -pi.z;
        L.wl = pi.w * 1.4426950408889634f;
    }
    // ---- once per solve: positions, Thole factors, staging indices; the operand slots start at 0
    if (t < N_DUMMY) {
        const float far = -2.0f * PHANTOM_FAR;
        s_a[count + t] = make_float4(far, far, far, 0.f);      // the dummy records follow the (only) chunk
        s_b[count + t] = make_float2(0.f, 0.f);
        s_w[count + t] = 0.f;
    }
    for (int l = t; l < count; l += GT) {
        const float4 p = a.stage_pos[gbase + l];
        s_idx[l] = ws.stage_atom[gbase + l];
        s_a[l] = make_float4(p.x, p.y, p.z, 0.f);
        s_b[l] = make_float2(0.f, 0.f);
        s_w[l] = p.w;
    }
    // the owner's atom in the caller's order; mu0 = alpha E or the caller's guess, published for the
    // first product (all CTAs gather it after the first grid barrier)
    double al = 0.0, ia = 0.0, E[3] = {0.0, 0.0, 0.0};
    const int atom = owner ? a.perm[slot] : -1;
    if (owner) {
        al = a.alpha_s[slot];
        ia = a.inv_alpha_s[slot];
        double m0[3] = {0.0, 0.0, 0.0};
        if (atom >= 0) {
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                E[k] = a.field[3 * (size_t)atom + k];
                m0[k] = a.use_guess ? a.mu[3 * (size_t)atom + k] : al * E[k];
            }
        }
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            s_vec[k * GT + t] = m0[k];
            s_p[k * GT + t] = 0.f;
        }
        a.mu0[slot] = make_float4((float)m0[0], (float)m0[1], (float)m0[2], 0.f);
    }
    unsigned gen = 0;
    if (a.test_fault && g == (int)gridDim.x - 1) return;      // tests: a CTA that is lost before the first barrier
    bool broken = !grid_barrier(st, gen);        // a barrier timed out: leave without touching the caller's mu
    double rz_old = 0.0, rr = 0.0;
    float delta = 0.f;
    int it = 0;                                  // iterations completed
    bool converged = false;

    for (int k = -1; k < a.max_iter && !broken; ++k) {
        // ---- operand: p_j <- u_j + delta p_j for every staged atom (k = -1: mu0; k = 0: delta = 0)
        __syncthreads();
        for (int l = t; l < count; l += GT) {
            const float4 u = __ldcg((k < 0 ? a.mu0 : a.u32) + s_idx[l]);
            float4 pa = s_a[l];
            float2 pb = s_b[l];
            pb.x = fmaf(delta, pb.x, u.x);
            pb.y = fmaf(delta, pb.y, u.y);
            pa.w = fmaf(delta, pa.w, u.z);
            s_a[l] = pa;
            s_b[l] = pb;
        }
        RowStream R;
        R.open(rows, t_total, part, wpb);
        __syncthreads();
        // ---- T v for my atom
        double dx = 0.0, dy = 0.0, dz = 0.0;
        if (active) {
            PartialTmu A;
            int d = 0, n_rows = 0, tg = part;
            int2 sd = seg[0];
            tmu_walk<FAR>(seg, 0, d, sd, tg, wpb, R, S, L, a.K, A, n_rows, dx, dy, dz);
            A.flush(dx, dy, dz, a.K.fixed);
            dx = acc_value(dx, a.K.fixed); dy = acc_value(dy, a.K.fixed); dz = acc_value(dz, a.K.fixed);
        }
        if (SPLIT && wpb > 1) {                    // uniform over the CTA: add the parts of a block, part 1 first
            __syncthreads();
            if (part > 0) {
                s_part[w * 96 + lane] = dx; s_part[w * 96 + 32 + lane] = dy; s_part[w * 96 + 64 + lane] = dz;
            }
            __syncthreads();
            if (part == 0)
                for (int q = 1; q < wpb; ++q) {
                    dx += s_part[(w + q) * 96 + lane]; dy += s_part[(w + q) * 96 + 32 + lane]; dz += s_part[(w + q) * 96 + 64 + lane];
                }
        }
        const double Tv[3] = {dx, dy, dz};
        double s1 = 0.0, s2 = 0.0;
        if (k < 0) {
            // r = E - (mu/alpha - T mu - self mu); u = alpha r; (r.z, r.r)
            if (owner) {
                float uf[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const double m = s_vec[c * GT + t];
                    const double r = E[c] - (m * ia - Tv[c] - a.self * m);
                    const double z = al * r;
                    s_vec[(3 + c) * GT + t] = r;
                    uf[c] = (float)z;
                    s1 += r * z; s2 += r * r;
                }
                a.u32[slot] = make_float4(uf[0], uf[1], uf[2], 0.f);
                s_p[t] = uf[0]; s_p[GT + t] = uf[1]; s_p[2 * GT + t] = uf[2];    // p0 = u (delta = 0)
            }
            block_sum2(s1, s2);
            if (t == 0) { a.part_a[2 * g] = s1; a.part_a[2 * g + 1] = s2; }
            if (!grid_barrier(st, gen)) { broken = true; break; }
            grid_totals(a.part_a, rz_old, rr);
            delta = 0.f;
            if (sqrt(rr / a.n_atoms) < a.tol) { converged = true; break; }
            continue;
        }
        // ---- q = p/alpha - T p - self p ; p.q
        double q[3] = {0, 0, 0}, p[3] = {0, 0, 0};
        if (owner) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                p[c] = (double)s_p[c * GT + t];
                q[c] = p[c] * ia - Tv[c] - a.self * p[c];
                s1 += p[c] * q[c];
            }
        }
        block_sum2(s1, s2);
        if (t == 0) { a.part_b[2 * g] = s1; a.part_b[2 * g + 1] = 0.0; }
        if (!grid_barrier(st, gen)) { broken = true; break; }
        double pq, unused;
        grid_totals(a.part_b, pq, unused);
        const double gamma = rz_old / pq;
        // ---- mu += gamma p ; r -= gamma q ; u = alpha r ; (r.z, r.r)
        s1 = 0.0; s2 = 0.0;
        float uf[3] = {0.f, 0.f, 0.f};
        if (owner) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                s_vec[c * GT + t] += gamma * p[c];
                const double r = s_vec[(3 + c) * GT + t] - gamma * q[c];
                s_vec[(3 + c) * GT + t] = r;
                const double z = al * r;
                uf[c] = (float)z;
                s1 += r * z; s2 += r * r;
            }
            a.u32[slot] = make_float4(uf[0], uf[1], uf[2], 0.f);
        }
        block_sum2(s1, s2);
        if (t == 0) { a.part_a[2 * g] = s1; a.part_a[2 * g + 1] = s2; }
        if (!grid_barrier(st, gen)) { broken = true; break; }
        double rz_new;
        grid_totals(a.part_a, rz_new, rr);
        it = k + 1;
        if (sqrt(rr / a.n_atoms) < a.tol) { converged = true; break; }
        delta = (float)(rz_new / rz_old);
        rz_old = rz_new;
        if (owner) {
#pragma unroll
            for (int c = 0; c < 3; ++c) s_p[c * GT + t] = fmaf(delta, s_p[c * GT + t], uf[c]);
        }
    }
    // ---- result, in the caller's order; the scalars go to host-mapped memory
    if (owner && atom >= 0 && !broken) {
#pragma unroll
        for (int c = 0; c < 3; ++c) a.mu[3 * (size_t)atom + c] = s_vec[c * GT + t];
    }
    if (g == 0 && t == 0) {
        st->rr = rr;
        st->iters = it;
        st->conv_at = converged ? it : 0x7fffffff;
        a.result[0] = rr;
        a.result[1] = (double)it;
        a.result[2] = broken ? 1.0 : 0.0;        // CTA 0 learns of a broken barrier no later than at its own next one
        __threadfence_system();
    }
}

// ----------------------------------------------------------------------------- host side
template <bool FAR, bool SPLIT>
static const void *persist_fn() { return (const void *)k_pcg_persist<FAR, SPLIT>; }

static const void *pick(Ctx *c, const ClusterWs &ws) {
    const bool split = c->n_blocks / ws.n_groups < 5;
    if (c->far_on) return split ? persist_fn<true, true>() : persist_fn<true, false>();
    return split ? persist_fn<false, true>() : persist_fn<false, false>();
}

int atom_solve_configure(Ctx *c) {
    const int big = 100 * 1024;
    TKHP_CUDA(c, cudaFuncSetAttribute(persist_fn<true, true>(), cudaFuncAttributeMaxDynamicSharedMemorySize, big));
    TKHP_CUDA(c, cudaFuncSetAttribute(persist_fn<true, false>(), cudaFuncAttributeMaxDynamicSharedMemorySize, big));
    TKHP_CUDA(c, cudaFuncSetAttribute(persist_fn<false, true>(), cudaFuncAttributeMaxDynamicSharedMemorySize, big));
    TKHP_CUDA(c, cudaFuncSetAttribute(persist_fn<false, false>(), cudaFuncAttributeMaxDynamicSharedMemorySize, big));
    int coop = 0;
    TKHP_CUDA(c, cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, c->p.device));
    c->coop_ok = coop != 0;
    return TKHP_OK;
}

// Can the persistent kernel run this solve?  (list header on the host: ensure_header has run)
bool atom_solve_eligible(Ctx *c) {
    if (!c->coop_ok || c->no_persist || c->stored_t || c->p.precision == TKHP_FP64 || c->list_mode_in_use != TKHP_LIST_ATOM) return false;
    ClusterWs ws = get_ws(c);
    const int s_max = atom_chunk_capacity(false, ws.chunk_cap);
    const int need = c->h_state->max_stage;
    if (need > s_max) return false;                        // some group needs more than one chunk
    const int s_chunk = (need + 31) & ~31;
    const size_t smem = solve_smem(s_chunk, c->n_blocks / ws.n_groups < 5);
    if (smem > 100 * 1024) return false;
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, pick(c, ws), GT, smem) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return (long long)per_sm * c->sm_count >= ws.n_groups && ws.n_groups <= c->part_cap;
}

// The kernel reads the field (and the guess) and writes mu in the caller's order; |r|^2, the iteration
// count and the barrier flag arrive in c->h_ring[0..2] (host-mapped) when the stream has drained.
int atom_solve_launch(Ctx *c, const double *d_field, double *d_mu, int use_guess, double tol, int max_iter, cudaStream_t s) {
    ClusterWs ws = get_ws(c);
    const double b = c->p.ewald_beta;
    SolveArgs a;
    a.ws = ws;
    a.gpos = ws.gpos32;
    a.stage_pos = ws.stage_pos32;
    a.mu0 = c->mu32;
    a.u32 = c->u32;
    a.K.pb = (float)((double)TKHP_ERFCX_P * b);
    a.K.nb2l = (float)(-1.4426950408889634 * b * b);
    a.K.c1b = (float)(2.0 / SQRT_PI * b);
    a.K.k3 = (float)(4.0 / (3.0 * SQRT_PI) * b * b * b);
    for (int k = 0; k < 6; ++k) a.K.q[k] = c->far_q[k];
    a.K.fixed = c->fixed ? 1 : 0;
    a.field = d_field;
    a.mu = d_mu;
    a.perm = c->perm;
    a.use_guess = use_guess;
    a.result = c->d_ring;
    a.alpha_s = c->alpha_s;
    a.inv_alpha_s = c->inv_alpha_s;
    a.part_a = c->partials;
    a.part_b = c->partials + 2 * (size_t)c->part_cap;
    a.st = c->st;
    a.tol = tol;
    a.self = 4.0 * b * b * b / (3.0 * SQRT_PI);
    a.max_iter = max_iter;
    a.n_atoms = c->n;
    a.n_pad = c->n_pad;
    a.s_chunk = (c->h_state->max_stage + 31) & ~31;
    a.rot_div = c->sm_count;
    a.test_fault = c->test_barrier_fault ? 1 : 0;
    TKHP_CUDA(c, cudaMemsetAsync(&c->st->bar_count, 0, 2 * sizeof(unsigned), s));
    void *args[] = {&a};
    if (cudaLaunchCooperativeKernel(pick(c, ws), dim3(ws.n_groups), dim3(GT), args, solve_smem(a.s_chunk, c->n_blocks / ws.n_groups < 5), s) != cudaSuccess)
        return set_err(c, TKHP_ECUDA, "cooperative launch of the persistent PCG kernel was refused%s");
    c->n_launches += 1;
    return TKHP_OK;
}

}  // namespace tkhp
