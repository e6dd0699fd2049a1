// pcg.cu -- everything around the pair kernels: packing to the sorted layout, the FP64
// mask-correction + self-term pass, the PCG vector kernels, the solve driver and the energy.
//
// Paper: "the polarization solver ... preconditioned conjugate gradient ... diagonal
// preconditioner" with one polarization matrix-vector product per iteration;
// scaling factors applied by a separate correction kernel over the few scaled pairs
// (Listing 2); energies need a DP container and a parallel (tree) reduction
// (P:L263-275).  Recurrences: DESIGN.md section 2 "S" (= SURVEY 8(c) S, Q10):
//   mu0 = alpha E (or the guess); r = E - A mu; z = alpha r; p = z;
//   loop: q = A p; gamma = (r.z)/(p.q); mu += gamma p; r -= gamma q; rms = sqrt(|r|^2/N);
//         z = alpha r; delta = (r.z)new/(r.z)old; p = z + delta p,     A v = v/alpha - T v.
// All vectors live in the SORTED, padded order (SoA x|y|z, FP64); dot products are FP64 two-level
// tree reductions (block partials, then every block of the next kernel re-reduces the partials:
// deterministic, no atomics, no extra launch).
#include "common.cuh"
#include "pair_math.cuh"

namespace tkhp {

constexpr int VEC_THREADS = 256;

// ----------------------------------------------------------------------------- packing
template <typename vec4>
__global__ void k_pack_mu_user(const double *__restrict__ mu, const int32_t *__restrict__ perm, int n_pad,
                               vec4 *__restrict__ out) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n_pad) return;
    int a = perm[s];
    double x = 0, y = 0, z = 0;
    if (a >= 0) { x = mu[3 * (size_t)a]; y = mu[3 * (size_t)a + 1]; z = mu[3 * (size_t)a + 2]; }
    vec4 v;
    v.x = x; v.y = y; v.z = z; v.w = 0;
    out[s] = v;
}

template <typename vec4>
__global__ void k_pack_multipoles(const double *__restrict__ q, const double *__restrict__ dip,
                                  const double *__restrict__ quad, const int32_t *__restrict__ group,
                                  const int32_t *__restrict__ perm, int n_pad, vec4 *__restrict__ mp) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n_pad) return;
    int a = perm[s];
    vec4 v0, v1, v2;
    v0.x = v0.y = v0.z = v0.w = 0;
    v1 = v0; v2 = v0;
    v2.z = -1 - (s & 31);   // phantoms: distinct negative "group"
    if (a >= 0) {
        v0.x = q[a];
        v0.y = dip[3 * (size_t)a]; v0.z = dip[3 * (size_t)a + 1]; v0.w = dip[3 * (size_t)a + 2];
        const double *t = quad + 6 * (size_t)a;
        v1.x = t[0]; v1.y = t[1]; v1.z = t[2]; v1.w = t[3];
        v2.x = t[4]; v2.y = t[5];
        v2.z = group[a];
    }
    mp[s] = v0; mp[n_pad + s] = v1; mp[2 * n_pad + s] = v2;
}

__global__ void k_tmatvec_finish(const double *__restrict__ acc, const int32_t *__restrict__ perm, int n_pad,
                                 const double *__restrict__ mu, double self, double *__restrict__ out) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n_pad) return;
    int a = perm[s];
    if (a < 0) return;
    for (int c = 0; c < 3; ++c)
        out[3 * (size_t)a + c] = acc[(size_t)c * n_pad + s] + self * mu[3 * (size_t)a + c];
}

// FP64 correction pass: adds, for every same-group pair within the cutoff, the masked field
// G_k = bn_k - rr_k (the tile/cluster kernels skip those pairs), plus the Ewald self term, and
// un-sorts the result.  One thread per atom walks its (few) group mates: "search, don't store"
// (P:L547).  Everything from the caller's FP64 inputs, minimum image per pair.
__global__ void k_field_finish(const double *__restrict__ acc, const int32_t *__restrict__ perm, int n_pad,
                               const double *__restrict__ pos, const int32_t *__restrict__ group,
                               const uint32_t *__restrict__ grp_start, const int32_t *__restrict__ grp_members,
                               const double *__restrict__ q, const double *__restrict__ dip,
                               const double *__restrict__ quad, double box, double beta, double rc2,
                               double self, double *__restrict__ field) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n_pad) return;
    const int a = perm[s];
    if (a < 0) return;
    double ex = acc[s], ey = acc[n_pad + s], ez = acc[2 * (size_t)n_pad + s];
    const int g = group[a];
    const double xa = pos[3 * (size_t)a], ya = pos[3 * (size_t)a + 1], za = pos[3 * (size_t)a + 2];
    for (uint32_t t = grp_start[g]; t < grp_start[g + 1]; ++t) {
        const int b = grp_members[t];
        if (b == a) continue;
        double Rx = xa - pos[3 * (size_t)b], Ry = ya - pos[3 * (size_t)b + 1], Rz = za - pos[3 * (size_t)b + 2];
        if (box > 0.0) {
            Rx -= box * rint(Rx / box); Ry -= box * rint(Ry / box); Rz -= box * rint(Rz / box);
        }
        const double r2 = Rx * Rx + Ry * Ry + Rz * Rz;
        if (r2 > rc2) continue;
        double G[3];
        radial_masked_f64(r2, beta, G);
        const double *d = dip + 3 * (size_t)b;
        const double *th = quad + 6 * (size_t)b;
        field_apply<double>(G, Rx, Ry, Rz, q[b], d[0], d[1], d[2], th[0], th[1], th[2], th[3], th[4], th[5],
                            ex, ey, ez);
    }
    field[3 * (size_t)a] = ex + self * dip[3 * (size_t)a];
    field[3 * (size_t)a + 1] = ey + self * dip[3 * (size_t)a + 1];
    field[3 * (size_t)a + 2] = ez + self * dip[3 * (size_t)a + 2];
}

// ----------------------------------------------------------------------------- reductions
// block-level sum of up to two values; result valid in thread 0
__device__ __forceinline__ void block_sum2(double &a, double &b) {
    __shared__ double sa[VEC_THREADS / 32], sb[VEC_THREADS / 32];
    a = warp_sum(a); b = warp_sum(b);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) { sa[w] = a; sb[w] = b; }
    __syncthreads();
    if (w == 0) {
        a = lane < VEC_THREADS / 32 ? sa[lane] : 0.0;
        b = lane < VEC_THREADS / 32 ? sb[lane] : 0.0;
        a = warp_sum(a); b = warp_sum(b);
    }
}

// every block re-reduces the partials of a previous kernel (fixed order => deterministic)
__device__ __forceinline__ void reduce_partials2(const double *__restrict__ part, int n_part, double &a, double &b) {
    __shared__ double bc[2];
    double x = 0, y = 0;
    for (int i = threadIdx.x; i < n_part; i += VEC_THREADS) { x += part[2 * i]; y += part[2 * i + 1]; }
    block_sum2(x, y);
    if (threadIdx.x == 0) { bc[0] = x; bc[1] = y; }
    __syncthreads();
    a = bc[0]; b = bc[1];
    __syncthreads();
}

template <typename vec4>
__device__ __forceinline__ void store_vec(vec4 *out, int s, double x, double y, double z) {
    vec4 v;
    v.x = x; v.y = y; v.z = z; v.w = 0;
    out[s] = v;
}

// ----------------------------------------------------------------------------- PCG kernels
// mu0 = alpha E or the guess; gather E to sorted order; pack mu for the first matvec
template <typename vec4>
__global__ void k_pcg_init(const double *__restrict__ field, const double *__restrict__ guess, int use_guess,
                           const int32_t *__restrict__ perm, const double *__restrict__ alpha_s, int n_pad,
                           double *__restrict__ vE, double *__restrict__ vmu, vec4 *__restrict__ packed) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n_pad) return;
    const int a = perm[s];
    double e[3] = {0, 0, 0}, m[3] = {0, 0, 0};
    if (a >= 0) {
        for (int c = 0; c < 3; ++c) {
            e[c] = field[3 * (size_t)a + c];
            m[c] = use_guess ? guess[3 * (size_t)a + c] : alpha_s[s] * e[c];
        }
    }
    for (int c = 0; c < 3; ++c) { vE[(size_t)c * n_pad + s] = e[c]; vmu[(size_t)c * n_pad + s] = m[c]; }
    store_vec(packed, s, m[0], m[1], m[2]);
}

// r = E - (mu/alpha - acc - self mu); z = alpha r; p = z; partials (r.z, r.r); pack p
template <typename vec4>
__global__ void k_pcg_residual0(const double *__restrict__ acc, const double *__restrict__ vE,
                                const double *__restrict__ vmu, const double *__restrict__ alpha_s,
                                const double *__restrict__ inv_alpha_s, double self, int n_pad,
                                double *__restrict__ vr, double *__restrict__ vp, vec4 *__restrict__ packed,
                                double *__restrict__ part_rz) {
    double rz = 0, rr = 0;
    for (int s = blockIdx.x * blockDim.x + threadIdx.x; s < n_pad; s += gridDim.x * blockDim.x) {
        const double al = alpha_s[s], ia = inv_alpha_s[s];
        double p[3];
        for (int c = 0; c < 3; ++c) {
            const size_t o = (size_t)c * n_pad + s;
            const double m = vmu[o];
            const double r = vE[o] - (m * ia - acc[o] - self * m);
            const double z = al * r;
            vr[o] = r; vp[o] = z; p[c] = z;
            rz += r * z; rr += r * r;
        }
        store_vec(packed, s, p[0], p[1], p[2]);
    }
    block_sum2(rz, rr);
    if (threadIdx.x == 0) { part_rz[2 * blockIdx.x] = rz; part_rz[2 * blockIdx.x + 1] = rr; }
}

// q = p/alpha - acc - self p ; partial p.q
__global__ void k_pcg_q(const double *__restrict__ acc, const double *__restrict__ vp,
                        const double *__restrict__ inv_alpha_s, double self, int n_pad, double *__restrict__ vq,
                        double *__restrict__ part_pq) {
    double pq = 0, dummy = 0;
    for (int s = blockIdx.x * blockDim.x + threadIdx.x; s < n_pad; s += gridDim.x * blockDim.x) {
        const double ia = inv_alpha_s[s];
        for (int c = 0; c < 3; ++c) {
            const size_t o = (size_t)c * n_pad + s;
            const double p = vp[o];
            const double q = p * ia - acc[o] - self * p;
            vq[o] = q;
            pq += p * q;
        }
    }
    block_sum2(pq, dummy);
    if (threadIdx.x == 0) { part_pq[2 * blockIdx.x] = pq; part_pq[2 * blockIdx.x + 1] = 0.0; }
}

// gamma = rz/pq ; mu += gamma p ; r -= gamma q ; partials (r.z, r.r) with z = alpha r
__global__ void k_pcg_update(const double *__restrict__ part_rz_old, const double *__restrict__ part_pq,
                             int n_part, const double *__restrict__ vp, const double *__restrict__ vq,
                             const double *__restrict__ alpha_s, int n_pad, double *__restrict__ vmu,
                             double *__restrict__ vr, double *__restrict__ part_rz_new) {
    double rz_old, rr_old, pq, dmy;
    reduce_partials2(part_rz_old, n_part, rz_old, rr_old);
    reduce_partials2(part_pq, n_part, pq, dmy);
    const double gamma = rz_old / pq;
    double rz = 0, rr = 0;
    for (int s = blockIdx.x * blockDim.x + threadIdx.x; s < n_pad; s += gridDim.x * blockDim.x) {
        const double al = alpha_s[s];
        for (int c = 0; c < 3; ++c) {
            const size_t o = (size_t)c * n_pad + s;
            vmu[o] += gamma * vp[o];
            const double r = vr[o] - gamma * vq[o];
            vr[o] = r;
            rz += r * (al * r); rr += r * r;
        }
    }
    block_sum2(rz, rr);
    if (threadIdx.x == 0) { part_rz_new[2 * blockIdx.x] = rz; part_rz_new[2 * blockIdx.x + 1] = rr; }
}

// delta = rz_new/rz_old ; p = alpha r + delta p ; pack p ; block 0 publishes |r|^2
template <typename vec4>
__global__ void k_pcg_direction(const double *__restrict__ part_rz_old, const double *__restrict__ part_rz_new,
                                int n_part, const double *__restrict__ vr, const double *__restrict__ alpha_s,
                                int n_pad, double *__restrict__ vp, vec4 *__restrict__ packed,
                                DeviceState *st) {
    double rz_old, rr_old, rz_new, rr_new;
    reduce_partials2(part_rz_old, n_part, rz_old, rr_old);
    reduce_partials2(part_rz_new, n_part, rz_new, rr_new);
    const double delta = rz_new / rz_old;
    if (blockIdx.x == 0 && threadIdx.x == 0) { st->rr = rr_new; st->rz = rz_new; st->delta = delta; }
    for (int s = blockIdx.x * blockDim.x + threadIdx.x; s < n_pad; s += gridDim.x * blockDim.x) {
        const double al = alpha_s[s];
        double p[3];
        for (int c = 0; c < 3; ++c) {
            const size_t o = (size_t)c * n_pad + s;
            p[c] = al * vr[o] + delta * vp[o];
            vp[o] = p[c];
        }
        store_vec(packed, s, p[0], p[1], p[2]);
    }
}

__global__ void k_publish_rr(const double *__restrict__ part_rz, int n_part, DeviceState *st) {
    double rz, rr;
    reduce_partials2(part_rz, n_part, rz, rr);
    if (threadIdx.x == 0) { st->rr = rr; st->rz = rz; }
}

__global__ void k_unsort3(const double *__restrict__ v, const int32_t *__restrict__ perm, int n_pad,
                          double *__restrict__ out) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n_pad) return;
    int a = perm[s];
    if (a < 0) return;
    for (int c = 0; c < 3; ++c) out[3 * (size_t)a + c] = v[(size_t)c * n_pad + s];
}

// ----------------------------------------------------------------------------- energy
__global__ void k_energy_partials(const double *__restrict__ mu, const double *__restrict__ field, long long n3,
                                  double *__restrict__ part) {
    double s = 0, dmy = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n3; i += (long long)gridDim.x * blockDim.x)
        s += mu[i] * field[i];
    block_sum2(s, dmy);
    if (threadIdx.x == 0) { part[2 * blockIdx.x] = s; part[2 * blockIdx.x + 1] = 0.0; }
}
__global__ void k_energy_final(const double *__restrict__ part, int n_part, double *__restrict__ energy) {
    double s, dmy;
    reduce_partials2(part, n_part, s, dmy);
    if (threadIdx.x == 0) *energy = -0.5 * COULOMB * s;
}

// ----------------------------------------------------------------------------- host drivers
static inline double self_coeff(const tkhp_params &p) {
    const double b = p.ewald_beta;
    return 4.0 * b * b * b / (3.0 * SQRT_PI);
}
static inline int vec_grid(const Ctx *c) {
    int g = div_up(c->n_pad, VEC_THREADS);
    return g < MAX_PARTIALS ? g : MAX_PARTIALS;
}

// live kernel timing: one event pair around the pair kernel alone (not the memset)
static inline bool prof_begin(Ctx *c, int which, cudaStream_t s) {
    if (!c->prof || c->prof_n[which] >= PROF_MAX) return false;
    cudaEventRecord(c->prof_ev[which][2 * c->prof_n[which]], s);
    return true;
}
static inline void prof_end(Ctx *c, int which, cudaStream_t s) {
    cudaEventRecord(c->prof_ev[which][2 * c->prof_n[which] + 1], s);
    c->prof_n[which]++;
}

int run_tmatvec(Ctx *c, cudaStream_t s) {
    // the tile kernel accumulates with atomics into zeroed accumulators; the cluster kernel stores
    if (c->list_mode_in_use == TKHP_LIST_TILES)
        TKHP_CUDA(c, cudaMemsetAsync(c->acc, 0, sizeof(double) * 3 * (size_t)c->n_pad, s));
    const bool rec = prof_begin(c, 0, s);
    int rc = c->list_mode_in_use == TKHP_LIST_ATOM      ? atom_tmatvec(c, s)
             : c->list_mode_in_use == TKHP_LIST_CLUSTER ? cluster_tmatvec(c, s)
                                                        : tiles_tmatvec(c, s);
    if (rec) prof_end(c, 0, s);
    return rc;
}
int run_field(Ctx *c, cudaStream_t s) {
    if (c->list_mode_in_use == TKHP_LIST_TILES)
        TKHP_CUDA(c, cudaMemsetAsync(c->acc, 0, sizeof(double) * 3 * (size_t)c->n_pad, s));
    const bool rec = prof_begin(c, 1, s);
    int rc = c->list_mode_in_use == TKHP_LIST_ATOM      ? atom_field(c, s)
             : c->list_mode_in_use == TKHP_LIST_CLUSTER ? cluster_field(c, s)
                                                        : tiles_field(c, s);
    if (rec) prof_end(c, 1, s);
    return rc;
}

int do_perm_field(Ctx *c, const double *d_q, const double *d_dip, const double *d_quad, double *d_field,
                  cudaStream_t s) {
    const int g = div_up(c->n_pad, VEC_THREADS);
    if (c->p.precision == TKHP_MIXED)
        k_pack_multipoles<float4><<<g, VEC_THREADS, 0, s>>>(d_q, d_dip, d_quad, c->group_o, c->perm, c->n_pad, c->mp32);
    else
        k_pack_multipoles<double4><<<g, VEC_THREADS, 0, s>>>(d_q, d_dip, d_quad, c->group_o, c->perm, c->n_pad, c->mp64);
    c->n_launches += 2;   // pack, finish
    int rc = run_field(c, s);
    if (rc) return rc;
    k_field_finish<<<g, VEC_THREADS, 0, s>>>(c->acc, c->perm, c->n_pad, c->pos_o, c->group_o, c->grp_start,
                                             c->grp_members, d_q, d_dip, d_quad, c->p.box, c->p.ewald_beta,
                                             c->p.cutoff * c->p.cutoff, self_coeff(c->p), d_field);
    TKHP_CUDA(c, cudaGetLastError());
    return TKHP_OK;
}

int do_tmatvec(Ctx *c, const double *d_mu, double *d_out, cudaStream_t s) {
    const int g = div_up(c->n_pad, VEC_THREADS);
    if (c->p.precision == TKHP_MIXED)
        k_pack_mu_user<float4><<<g, VEC_THREADS, 0, s>>>(d_mu, c->perm, c->n_pad, c->mu32);
    else
        k_pack_mu_user<double4><<<g, VEC_THREADS, 0, s>>>(d_mu, c->perm, c->n_pad, c->mu64);
    c->n_launches += 2;   // pack, finish
    int rc = run_tmatvec(c, s);
    if (rc) return rc;
    k_tmatvec_finish<<<g, VEC_THREADS, 0, s>>>(c->acc, c->perm, c->n_pad, d_mu, self_coeff(c->p), d_out);
    TKHP_CUDA(c, cudaGetLastError());
    return TKHP_OK;
}

static int read_rr(Ctx *c, cudaStream_t s, double *rr) {
    TKHP_CUDA(c, cudaMemcpyAsync(c->h_scalars, &c->st->rr, sizeof(double), cudaMemcpyDeviceToHost, s));
    TKHP_CUDA(c, cudaStreamSynchronize(s));
    *rr = c->h_scalars[0];
    return TKHP_OK;
}

int do_polar_solve(Ctx *c, const double *d_field, double *d_mu, double tol, int max_iter, int use_guess,
                   int *h_iters, double *h_rms, cudaStream_t s) {
    const int n_pad = c->n_pad;
    const int g1 = div_up(n_pad, VEC_THREADS);
    const int gv = vec_grid(c);
    const double self = self_coeff(c->p);
    const bool mixed = c->p.precision == TKHP_MIXED;
    double *part_rz[2] = {c->partials, c->partials + 2 * MAX_PARTIALS};
    double *part_pq = c->partials + 4 * MAX_PARTIALS;
    int rc;

    if (mixed)
        k_pcg_init<float4><<<g1, VEC_THREADS, 0, s>>>(d_field, d_mu, use_guess, c->perm, c->alpha_s, n_pad, c->vE, c->vmu, c->mu32);
    else
        k_pcg_init<double4><<<g1, VEC_THREADS, 0, s>>>(d_field, d_mu, use_guess, c->perm, c->alpha_s, n_pad, c->vE, c->vmu, c->mu64);
    if ((rc = run_tmatvec(c, s))) return rc;
    if (mixed)
        k_pcg_residual0<float4><<<gv, VEC_THREADS, 0, s>>>(c->acc, c->vE, c->vmu, c->alpha_s, c->inv_alpha_s, self, n_pad, c->vr, c->vp, c->mu32, part_rz[0]);
    else
        k_pcg_residual0<double4><<<gv, VEC_THREADS, 0, s>>>(c->acc, c->vE, c->vmu, c->alpha_s, c->inv_alpha_s, self, n_pad, c->vr, c->vp, c->mu64, part_rz[0]);
    k_publish_rr<<<1, VEC_THREADS, 0, s>>>(part_rz[0], gv, c->st);
    c->n_launches += 3;   // init, residual0, publish
    double rr;
    if ((rc = read_rr(c, s, &rr))) return rc;
    double rms = sqrt(rr / c->n);
    int it = 0;
    while (rms >= tol && it < max_iter) {
        const int cur = it & 1, nxt = cur ^ 1;
        if ((rc = run_tmatvec(c, s))) return rc;
        k_pcg_q<<<gv, VEC_THREADS, 0, s>>>(c->acc, c->vp, c->inv_alpha_s, self, n_pad, c->vq, part_pq);
        k_pcg_update<<<gv, VEC_THREADS, 0, s>>>(part_rz[cur], part_pq, gv, c->vp, c->vq, c->alpha_s, n_pad, c->vmu, c->vr, part_rz[nxt]);
        if (mixed)
            k_pcg_direction<float4><<<gv, VEC_THREADS, 0, s>>>(part_rz[cur], part_rz[nxt], gv, c->vr, c->alpha_s, n_pad, c->vp, c->mu32, c->st);
        else
            k_pcg_direction<double4><<<gv, VEC_THREADS, 0, s>>>(part_rz[cur], part_rz[nxt], gv, c->vr, c->alpha_s, n_pad, c->vp, c->mu64, c->st);
        c->n_launches += 3;   // q, update, direction
        ++it;
        if ((rc = read_rr(c, s, &rr))) return rc;
        rms = sqrt(rr / c->n);
        if (!(rms == rms)) break;   // NaN: give up
    }
    k_unsort3<<<g1, VEC_THREADS, 0, s>>>(c->vmu, c->perm, n_pad, d_mu);
    c->n_launches += 1;
    TKHP_CUDA(c, cudaGetLastError());
    TKHP_CUDA(c, cudaStreamSynchronize(s));
    if (h_iters) *h_iters = it;
    if (h_rms) *h_rms = rms;
    if (!(rms < tol)) return set_err(c, TKHP_ENOCONV, "PCG did not reach the tolerance within max_iter%s");
    return TKHP_OK;
}

int do_polar_energy(Ctx *c, const double *d_mu, const double *d_field, double *d_energy, cudaStream_t s) {
    const long long n3 = 3LL * c->n;
    int g = div_up(n3, VEC_THREADS);
    if (g > MAX_PARTIALS) g = MAX_PARTIALS;
    double *part = c->partials + 6 * MAX_PARTIALS;
    k_energy_partials<<<g, VEC_THREADS, 0, s>>>(d_mu, d_field, n3, part);
    k_energy_final<<<1, VEC_THREADS, 0, s>>>(part, g, d_energy);
    c->n_launches += 2;
    TKHP_CUDA(c, cudaGetLastError());
    return TKHP_OK;
}

}  // namespace tkhp
