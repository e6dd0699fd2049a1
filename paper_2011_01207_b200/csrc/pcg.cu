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
// tree reductions (block partials, then the last block of the same kernel re-reduces them in a
// fixed order: deterministic, no floating-point atomics, no extra launch; reduce.cuh).
#include "common.cuh"
#include "pair_math.cuh"
#include "reduce.cuh"

namespace tkhp {

constexpr int VEC_THREADS = RED_THREADS;

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
        if (r2 > rc2 || r2 <= 1e-20) continue;              // (coincident group mates: no 1/0)
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

template <typename vec4>
__device__ __forceinline__ void store_vec(vec4 *out, int s, double x, double y, double z) {
    vec4 v;
    v.x = x; v.y = y; v.z = z; v.w = 0;
    out[s] = v;
}

// ----------------------------------------------------------------------------- PCG kernels
// Device-side control (no host round trip per iteration): st->conv_at = first iteration index that
// must NOT run; every kernel of iteration `iter` returns at once when iter >= conv_at.  The kernel
// that forms a new residual (k_pcg_residual0, k_pcg_update) lowers conv_at in its last block, i.e.
// after every block of that kernel has passed its own test.
//
// mu0 = alpha E or the guess; gather E to sorted order; pack mu for the first matvec
template <typename vec4>
__global__ void k_pcg_init(const double *__restrict__ field, const double *__restrict__ guess, int use_guess,
                           const int32_t *__restrict__ perm, const double *__restrict__ alpha_s, int n_pad,
                           double *__restrict__ vE, double *__restrict__ vmu, vec4 *__restrict__ packed,
                           DeviceState *st) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s == 0) { st->conv_at = 0x7fffffff; st->iters = 0; st->ticket = 0u; st->bar_gen = -1; }
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

// r = E - (mu/alpha - acc - self mu); z = alpha r; p = z; (r.z, r.r) -> st->rzv[0], ring slot 0; pack p
template <typename vec4>
__global__ void __launch_bounds__(RED_THREADS)
k_pcg_residual0(const double *__restrict__ acc, const double *__restrict__ vE, const double *__restrict__ vmu,
                const double *__restrict__ alpha_s, const double *__restrict__ inv_alpha_s, double self, int n_pad,
                double *__restrict__ vr, double *__restrict__ vp, vec4 *__restrict__ packed,
                double *__restrict__ part, DeviceState *st, double tol, int n_atoms, volatile double *ring_slot) {
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
    if (grid_sum2_last_block(part, &st->ticket, rz, rr) && threadIdx.x == 0)
        pcg_publish_residual(st, 0, rz, rr, 0, tol, n_atoms, ring_slot);
}

// q = p/alpha - acc - self p ; p.q -> st->pq   (TILES and CLUSTER modes; the ATOM-mode pair kernel
// does this in its epilogue)
__global__ void __launch_bounds__(RED_THREADS)
k_pcg_q(const double *__restrict__ acc, const double *__restrict__ vp, const double *__restrict__ inv_alpha_s,
        double self, int n_pad, double *__restrict__ vq, double *__restrict__ part, DeviceState *st, int iter) {
    if (iter >= st->conv_at) return;
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
    if (grid_sum2_last_block(part, &st->ticket, pq, dummy) && threadIdx.x == 0) st->pq = pq;
}

// gamma = rz/pq ; mu += gamma p ; r -= gamma q ; (r.z, r.r) with z = alpha r -> st->rzv[nxt], ring
__global__ void __launch_bounds__(RED_THREADS)
k_pcg_update(const double *__restrict__ vp, const double *__restrict__ vq, const double *__restrict__ alpha_s,
             int n_pad, double *__restrict__ vmu, double *__restrict__ vr, double *__restrict__ part,
             DeviceState *st, int iter, double tol, int n_atoms, volatile double *ring_slot) {
    if (iter >= st->conv_at) return;
    const double gamma = st->rzv[iter & 1] / st->pq;
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
    if (grid_sum2_last_block(part, &st->ticket, rz, rr) && threadIdx.x == 0)
        pcg_publish_residual(st, (iter + 1) & 1, rz, rr, iter + 1, tol, n_atoms, ring_slot);
}

// delta = rz_new/rz_old ; p = alpha r + delta p ; pack p   (not needed once converged)
template <typename vec4>
__global__ void k_pcg_direction(const double *__restrict__ vr, const double *__restrict__ alpha_s, int n_pad,
                                double *__restrict__ vp, vec4 *__restrict__ packed,
                                const DeviceState *__restrict__ st, int iter) {
    if (iter + 1 >= st->conv_at) return;
    const double delta = st->rzv[(iter + 1) & 1] / st->rzv[iter & 1];
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

// One PCG iteration's vector work in ONE cooperative launch (all blocks resident): the update
// (gamma = rz/pq; mu += gamma p; r -= gamma q; partial r.z, r.r), a grid barrier, then the direction
// (delta = rz_new/rz_old; p = alpha r + delta p; pack p) from the r, alpha and p still in registers.
// Every block adds the partial sums of all blocks in the same order, so all of them hold identical
// totals and take the same convergence decision; block 0 publishes.  Replaces k_pcg_update +
// k_pcg_direction: one launch and one pass over r, alpha, p less per iteration.  One atom per thread.
template <typename vec4>
__global__ void __launch_bounds__(RED_THREADS)
k_pcg_step(double *__restrict__ vp, const double *__restrict__ vq, const double *__restrict__ alpha_s, int n_pad,
           double *__restrict__ vmu, double *__restrict__ vr, vec4 *__restrict__ packed, double *__restrict__ part,
           DeviceState *st, int iter, double tol, int n_atoms, volatile double *ring_slot) {
    if (iter >= st->conv_at) return;
    const double rz_old = st->rzv[iter & 1];
    const double gamma = rz_old / st->pq;
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    double al = 0.0, r[3] = {0, 0, 0}, p[3] = {0, 0, 0};
    double rz = 0, rr = 0;
    if (s < n_pad) {
        al = alpha_s[s];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const size_t o = (size_t)c * n_pad + s;
            p[c] = vp[o];
            vmu[o] += gamma * p[c];
            r[c] = vr[o] - gamma * vq[o];
            vr[o] = r[c];
            rz += r[c] * (al * r[c]); rr += r[c] * r[c];
        }
    }
    block_sum2(rz, rr);
    // ---- grid barrier: partials out, last arriver opens the gate for this iteration
    __shared__ double s_tot[2];
    if (threadIdx.x == 0) {
        part[2 * blockIdx.x] = rz;
        part[2 * blockIdx.x + 1] = rr;
        __threadfence();
        if (atomicInc(&st->ticket, gridDim.x - 1) == gridDim.x - 1) {
            __threadfence();
            *reinterpret_cast<volatile int *>(&st->bar_gen) = iter;
        } else {
            while (*reinterpret_cast<volatile int *>(&st->bar_gen) != iter) {}
        }
        __threadfence();
    }
    __syncthreads();
    double x = 0, y = 0;
    for (int i = threadIdx.x; i < (int)gridDim.x; i += RED_THREADS) {
        x += __ldcg(part + 2 * i);
        y += __ldcg(part + 2 * i + 1);
    }
    block_sum2(x, y);
    if (threadIdx.x == 0) { s_tot[0] = x; s_tot[1] = y; }
    __syncthreads();
    const double rz_new = s_tot[0], rr_new = s_tot[1];
    const bool converged = sqrt(rr_new / n_atoms) < tol;      // same test as the host's: no new direction then
    if (!converged && s < n_pad) {
        const double delta = rz_new / rz_old;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            p[c] = al * r[c] + delta * p[c];
            vp[(size_t)c * n_pad + s] = p[c];
        }
        store_vec(packed, s, p[0], p[1], p[2]);
    }
    // the scalars and the host's copy of |r|^2 last: the system-scope fence of the publish is off the
    // other blocks' path and behind block 0's own stores
    if (blockIdx.x == 0 && threadIdx.x == 0)
        pcg_publish_residual(st, (iter + 1) & 1, rz_new, rr_new, iter + 1, tol, n_atoms, ring_slot);
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
__global__ void __launch_bounds__(RED_THREADS)
k_energy(const double *__restrict__ mu, const double *__restrict__ field, long long n3, double *__restrict__ part,
         DeviceState *st, double *__restrict__ energy) {
    double s = 0, dmy = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n3; i += (long long)gridDim.x * blockDim.x)
        s += mu[i] * field[i];
    block_sum2(s, dmy);
    if (grid_sum2_last_block(part, &st->ticket, s, dmy) && threadIdx.x == 0) *energy = -0.5 * COULOMB * s;
}

// TKHP_FIXED (Q21): every ATOM's term -1/2 f mu_i.E_i goes into an int64 container
// with 30 fractional bits (kcal/mol) -- one conversion per atom, of the dot product ((x + y) + z) formed
// without fused multiply-adds, so that the integer is a defined function of the inputs.  Integer sums do not
// depend on the order, so warp sums and one integer atomic per warp are deterministic.  The last block
// converts back (eq. 3) and clears the container.  __double2ll_rn saturates: a term of 2^33 kcal/mol or more
// cannot be held (the paper's mode has no guard against that either).
__global__ void __launch_bounds__(RED_THREADS)
k_energy_fixed(const double *__restrict__ mu, const double *__restrict__ field, long long n_atoms, DeviceState *st,
               double *__restrict__ energy) {
    long long s = 0;
    const double scale = -0.5 * COULOMB * (double)(1ll << FIX_ENERGY_BITS);
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_atoms; i += (long long)gridDim.x * blockDim.x) {
        const double *m = mu + 3 * i, *e = field + 3 * i;
        const double dot = __dadd_rn(__dadd_rn(__dmul_rn(m[0], e[0]), __dmul_rn(m[1], e[1])), __dmul_rn(m[2], e[2]));
        s += __double2ll_rn(__dmul_rn(dot, scale));
    }
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) atomicAdd(&st->energy_fixed, (unsigned long long)s);
    __shared__ bool s_last;
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        s_last = atomicInc(&st->ticket, gridDim.x - 1) == gridDim.x - 1;
    }
    __syncthreads();
    if (s_last && threadIdx.x == 0) {
        __threadfence();
        const long long tot = (long long)atomicExch(&st->energy_fixed, 0ull);
        *energy = (double)tot * (1.0 / (double)(1ll << FIX_ENERGY_BITS));
    }
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
    c->prof_iter[which][c->prof_n[which]] = c->spec_iter;
    c->prof_skip[which][c->prof_n[which]] = false;
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
    if (c->p.precision != TKHP_FP64)
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
    if (c->p.precision != TKHP_FP64)
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

// Wait for the device to publish |r|^2 into a ring slot (mapped pinned memory).  The host spins on
// the slot; every few thousand spins it asks the stream whether it failed or drained (a drained
// stream with an untouched slot means a kernel died).
static int wait_slot(Ctx *c, cudaStream_t s, int slot, double *rr) {
    volatile double *v = c->h_ring + slot;
    for (unsigned spin = 1;; ++spin) {
        const double x = *v;
        if (!(x == -1.0)) { *rr = x; return TKHP_OK; }
        if ((spin & 0xfff) == 0) {
            const cudaError_t e = cudaStreamQuery(s);
            if (e == cudaSuccess) {
                const double y = *v;
                if (!(y == -1.0)) { *rr = y; return TKHP_OK; }
                return set_err(c, TKHP_ECUDA, "PCG residual was never published%s");
            }
            if (e != cudaErrorNotReady) TKHP_CUDA(c, e);
        }
    }
}

// The solve runs without a host round trip per iteration: the host enqueues iterations up to
// PCG_LAG ahead of the last residual it has seen; the direction kernel of iteration k publishes
// |r|^2 to the ring and lowers st->conv_at to k + 1 when rms < tol, which turns every kernel of
// later (speculatively enqueued) iterations into an immediate return.
int do_polar_solve(Ctx *c, const double *d_field, double *d_mu, double tol, int max_iter, int use_guess,
                   int *h_iters, double *h_rms, cudaStream_t s) {
    const int n_pad = c->n_pad;
    const int g1 = div_up(n_pad, VEC_THREADS);
    const int gv = vec_grid(c);
    const double self = self_coeff(c->p);
    const bool mixed = c->p.precision != TKHP_FP64;
    double *part_rz = c->partials;
    double *part_pq = c->partials + 2 * (size_t)c->part_cap;
    const bool fused_q = c->list_mode_in_use == TKHP_LIST_ATOM;   // q and p.q in the pair kernel's epilogue
    int rc;
    // the fused update+direction kernel has a grid barrier: one atom per thread and every block resident
    bool fused_step = false;
    {
        int per_sm = 0;
        const void *fn = mixed ? (const void *)k_pcg_step<float4> : (const void *)k_pcg_step<double4>;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, VEC_THREADS, 0) == cudaSuccess)
            fused_step = c->coop_ok && !c->no_fused_step && g1 <= per_sm * c->sm_count && g1 <= c->part_cap;
        else
            cudaGetLastError();
    }

    // ---- the whole solve as one persistent cooperative kernel (atom_solve.cu) when it can run: it
    // reads the field and the guess and writes mu in the caller's order, the scalars come back
    // through host-mapped memory
    const bool persist_atom = atom_solve_eligible(c);
    if (persist_atom || tiles_solve_eligible(c)) {
        const bool rec = c->prof && c->prof_n[2] < PROF_MAX;
        if (rec) cudaEventRecord(c->prof_ev[2][2 * c->prof_n[2]], s);
        rc = persist_atom ? atom_solve_launch(c, d_field, d_mu, use_guess, tol, max_iter, s)
                          : tiles_solve_launch(c, d_field, d_mu, use_guess, tol, max_iter, s);
        if (rec) { cudaEventRecord(c->prof_ev[2][2 * c->prof_n[2] + 1], s); c->prof_n[2]++; }
        const cudaError_t e = cudaStreamSynchronize(s);
        if (rc == TKHP_ECUDA && e == cudaSuccess) {
            // the cooperative launch itself was refused: launch-per-matvec path, now and later
            cudaGetLastError();
            c->no_persist = true;
            if (rec) c->prof_n[2]--;
            return do_polar_solve(c, d_field, d_mu, tol, max_iter, use_guess, h_iters, h_rms, s);
        }
        if (rc) return rc;
        TKHP_CUDA(c, e);
        const int it_done = (int)c->h_ring[1];
        const double rms_done = sqrt(c->h_ring[0] / c->n);
        if (c->h_ring[2] != 0.0) {
            // A grid barrier of the persistent kernel timed out (a CTA never arrived within 2 s).  The kernel left
            // d_mu as the caller passed it, so nothing is lost: this context stops using persistent kernels and the
            // solve is repeated on the launch-per-matvec path.
            c->no_persist = true;
            c->n_barrier_timeouts += 1;
            if (rec) c->prof_n[2]--;
            return do_polar_solve(c, d_field, d_mu, tol, max_iter, use_guess, h_iters, h_rms, s);
        }
        if (rec) c->prof_solve_matvecs += it_done + 1;
        if (h_iters) *h_iters = it_done;
        if (h_rms) *h_rms = rms_done;
        if (!(rms_done < tol)) return set_err(c, TKHP_ENOCONV, "PCG did not reach the tolerance within max_iter%s");
        return TKHP_OK;
    }

    for (int k = 0; k < RING; ++k) c->h_ring[k] = -1.0;
    const int prof_first = c->prof_n[0];
    if (mixed)
        k_pcg_init<float4><<<g1, VEC_THREADS, 0, s>>>(d_field, d_mu, use_guess, c->perm, c->alpha_s, n_pad, c->vE, c->vmu, c->mu32, c->st);
    else
        k_pcg_init<double4><<<g1, VEC_THREADS, 0, s>>>(d_field, d_mu, use_guess, c->perm, c->alpha_s, n_pad, c->vE, c->vmu, c->mu64, c->st);
    c->spec_iter = -1;
    if ((rc = run_tmatvec(c, s))) return rc;
    if (mixed)
        k_pcg_residual0<float4><<<gv, VEC_THREADS, 0, s>>>(c->acc, c->vE, c->vmu, c->alpha_s, c->inv_alpha_s, self, n_pad, c->vr, c->vp, c->mu32, part_rz, c->st, tol, c->n, c->d_ring);
    else
        k_pcg_residual0<double4><<<gv, VEC_THREADS, 0, s>>>(c->acc, c->vE, c->vmu, c->alpha_s, c->inv_alpha_s, self, n_pad, c->vr, c->vp, c->mu64, part_rz, c->st, tol, c->n, c->d_ring);
    c->n_launches += 2;   // init, residual0

    // result j = |r|^2 after j iterations, in ring slot j % RING
    int enq = 0, seen = 0, it = 0;
    double rr = 0.0, rms = 0.0;
    for (;;) {
        while (enq < max_iter && enq < seen + PCG_LAG) {
            const int slot = (enq + 1) % RING;
            c->h_ring[slot] = -1.0;                 // consumed PCG_LAG < RING results ago
            c->spec_iter = enq;
            c->fuse_q = fused_q;
            rc = run_tmatvec(c, s);
            c->spec_iter = -1;
            c->fuse_q = false;
            if (rc) { cudaStreamSynchronize(s); return rc; }
            if (!fused_q) {
                k_pcg_q<<<gv, VEC_THREADS, 0, s>>>(c->acc, c->vp, c->inv_alpha_s, self, n_pad, c->vq, part_pq, c->st, enq);
                c->n_launches += 1;
            }
            if (fused_step) {
                // one cooperative launch: update, grid barrier, direction (k_pcg_step)
                double *a_vp = c->vp; const double *a_vq = c->vq; const double *a_al = c->alpha_s; int a_n = n_pad;
                double *a_mu = c->vmu; double *a_r = c->vr; void *a_pk = mixed ? (void *)c->mu32 : (void *)c->mu64;
                double *a_part = part_rz; DeviceState *a_st = c->st; int a_it = enq; double a_tol = tol; int a_na = c->n;
                volatile double *a_ring = c->d_ring + slot;
                void *args[] = {&a_vp, &a_vq, &a_al, &a_n, &a_mu, &a_r, &a_pk, &a_part, &a_st, &a_it, &a_tol, &a_na, &a_ring};
                const void *fn = mixed ? (const void *)k_pcg_step<float4> : (const void *)k_pcg_step<double4>;
                if (cudaLaunchCooperativeKernel(fn, dim3(g1), dim3(VEC_THREADS), args, 0, s) == cudaSuccess) {
                    c->n_launches += 1;
                } else {
                    // e.g. cudaErrorCooperativeLaunchTooLarge under MPS / SM partitioning: the two-kernel
                    // form from this iteration on (nothing of this iteration has been enqueued yet)
                    cudaGetLastError();
                    fused_step = false;
                    c->no_fused_step = true;
                }
            }
            if (!fused_step) {
                k_pcg_update<<<gv, VEC_THREADS, 0, s>>>(c->vp, c->vq, c->alpha_s, n_pad, c->vmu, c->vr, part_rz, c->st, enq, tol, c->n, c->d_ring + slot);
                if (mixed)
                    k_pcg_direction<float4><<<gv, VEC_THREADS, 0, s>>>(c->vr, c->alpha_s, n_pad, c->vp, c->mu32, c->st, enq);
                else
                    k_pcg_direction<double4><<<gv, VEC_THREADS, 0, s>>>(c->vr, c->alpha_s, n_pad, c->vp, c->mu64, c->st, enq);
                c->n_launches += 2;   // update, direction
            }
            ++enq;
        }
        if ((rc = wait_slot(c, s, seen % RING, &rr))) { cudaStreamSynchronize(s); return rc; }
        it = seen++;                                // iterations completed when this residual was formed
        rms = sqrt(rr / c->n);
        if (rms < tol || !(rms == rms) || it >= max_iter) break;
    }
    // speculative iterations enqueued after convergence returned at once: keep them out of the counts
    if (rms < tol) {
        if (fused_step) c->n_noop_launches += (fused_q ? 2LL : 3LL) * (enq - it);
        else c->n_noop_launches += (fused_q ? 3LL : 4LL) * (enq - it) + (it > 0 ? 1 : 0);   // + the last direction
        for (int i = prof_first; i < c->prof_n[0]; ++i)
            if (c->prof_iter[0][i] >= it) c->prof_skip[0][i] = true;
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
    double *part = c->partials + 4 * (size_t)c->part_cap;
    if (c->fixed) k_energy_fixed<<<g, VEC_THREADS, 0, s>>>(d_mu, d_field, (long long)c->n, c->st, d_energy);
    else k_energy<<<g, VEC_THREADS, 0, s>>>(d_mu, d_field, n3, part, c->st, d_energy);
    c->n_launches += 1;
    TKHP_CUDA(c, cudaGetLastError());
    return TKHP_OK;
}

}  // namespace tkhp
