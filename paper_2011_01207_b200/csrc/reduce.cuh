// reduce.cuh -- deterministic FP64 dot-product reductions for the PCG kernels.
//
// Paper: energies and dot products need a 64-bit container and a parallel (tree) reduction
// (P:L263-275).  Every kernel that produces a dot product writes one partial per block; the LAST
// block to finish (ticket counter) re-reduces all partials in a fixed order and stores the scalar
// in DeviceState, so that the next kernel reads one number.  No floating-point atomics: the result
// does not depend on the order in which blocks finish.
#pragma once
#include "common.cuh"

namespace tkhp {

constexpr int RED_THREADS = 256;      // block size of every kernel that uses these helpers

// block-level sum of two values; result valid in thread 0
__device__ __forceinline__ void block_sum2(double &a, double &b) {
    __shared__ double sa[RED_THREADS / 32], sb[RED_THREADS / 32];
    a = warp_sum(a); b = warp_sum(b);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) { sa[w] = a; sb[w] = b; }
    __syncthreads();
    if (w == 0) {
        a = lane < RED_THREADS / 32 ? sa[lane] : 0.0;
        b = lane < RED_THREADS / 32 ? sb[lane] : 0.0;
        a = warp_sum(a); b = warp_sum(b);
    }
}

// Called by ALL threads of every block of the grid with the block's two partial sums (valid in
// thread 0).  Returns true in all threads of the last block, with the grid totals in a, b (valid in
// thread 0 of that block).  `ticket` returns to 0 for the next kernel.
__device__ __forceinline__ bool grid_sum2_last_block(double *__restrict__ part, unsigned *ticket, double &a, double &b) {
    __shared__ bool s_last;
    const int n_part = gridDim.x;
    if (threadIdx.x == 0) {
        part[2 * blockIdx.x] = a;
        part[2 * blockIdx.x + 1] = b;
        __threadfence();
        s_last = atomicInc(ticket, (unsigned)(n_part - 1)) == (unsigned)(n_part - 1);
    }
    __syncthreads();
    if (!s_last) return false;
    __threadfence();
    double x = 0, y = 0;
    for (int i = threadIdx.x; i < n_part; i += RED_THREADS) {
        x += __ldcg(part + 2 * i);
        y += __ldcg(part + 2 * i + 1);
    }
    block_sum2(x, y);
    a = x; b = y;
    return true;
}

// |r|^2 of one PCG iteration into the host-mapped ring (the host polls the slot: no copy, no sync)
__device__ __forceinline__ void publish(volatile double *ring_slot, double rr) {
    *ring_slot = rr;
    __threadfence_system();
}

// Last-block epilogue of the kernels that produce the new residual: scalars, convergence, ring.
__device__ __forceinline__ void pcg_publish_residual(DeviceState *st, int which, double rz, double rr, int iter_done,
                                                     double tol, int n_atoms, volatile double *ring_slot) {
    st->rzv[which] = rz;
    st->rr = rr;
    st->iters = iter_done;
    if (sqrt(rr / n_atoms) < tol) st->conv_at = iter_done;       // same expression as the host's test
    publish(ring_slot, rr);
}

// ---- grid-wide barrier and totals of the persistent PCG kernels (cooperative launch: all CTAs resident)
__device__ __forceinline__ unsigned ld_acquire(const unsigned *p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long global_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
constexpr unsigned BAR_POISON = 0x80000000u;                 // bit 31 of bar_count: some CTA gave up waiting
constexpr unsigned long long BAR_TIMEOUT_NS = 2000000000ull; // 2 s of %globaltimer, whatever the clocks are

// All threads of all CTAs.  `gen` counts the barriers this CTA has passed.  One atomic per CTA on a
// counter that only grows during a solve; everybody spins on the counter itself (one L2 round trip
// less on the critical path than a separate release word written by the last arriver).
// Returns false (uniformly over the CTA) when the barrier is broken: a CTA that has waited for
// BAR_TIMEOUT_NS sets bit 31 of the counter, which every other CTA sees in the value it polls or in
// the value its own arrival returns -- at this barrier or at its next one, with no extra memory
// access on the good path.  After `false` the partial sums are inconsistent: the caller must leave
// its loop without writing results.  (The arrival counts stay far below 2^31: barriers per solve x CTAs.)
__device__ __forceinline__ bool grid_barrier(DeviceState *st, unsigned &gen) {
    int bad = 0;
    __syncthreads();
    ++gen;
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned target = gen * gridDim.x;
        unsigned v = atomicAdd(&st->bar_count, 1u) + 1u;
        if (v < target) {
            unsigned long long t0 = 0;
            for (unsigned n = 1; (v = ld_acquire(&st->bar_count)) < target; ++n) {
                if ((n & 0x3ffu) != 0) continue;                      // look at the clock every 1024 polls
                const unsigned long long now = global_ns();
                if (t0 == 0) t0 = now;
                else if (now - t0 > BAR_TIMEOUT_NS) {
                    v = atomicOr(&st->bar_count, BAR_POISON) | BAR_POISON;
                    st->err_barrier = 1;
                    break;
                }
            }
        }
        bad = (v & BAR_POISON) != 0u;
        __threadfence();
    }
    return __syncthreads_or(bad) == 0;      // the closing CTA barrier also hands thread 0's verdict to everybody
}

// identical in every CTA: sum of the per-CTA partials in a fixed order
__device__ __forceinline__ void grid_totals(const double *part, double &a, double &b) {
    __shared__ double s_tot[2];
    double x = 0, y = 0;
    for (int i = threadIdx.x; i < (int)gridDim.x; i += RED_THREADS) {
        x += __ldcg(part + 2 * i);
        y += __ldcg(part + 2 * i + 1);
    }
    block_sum2(x, y);
    if (threadIdx.x == 0) { s_tot[0] = x; s_tot[1] = y; }
    __syncthreads();
    a = s_tot[0]; b = s_tot[1];
}

}  // namespace tkhp
