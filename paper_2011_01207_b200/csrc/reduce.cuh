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
// All threads of all CTAs.  `gen` counts the barriers this CTA has passed.  One atomic per CTA on a
// counter that only grows during a solve; everybody spins on the counter itself (one L2 round trip
// less on the critical path than a separate release word written by the last arriver).
__device__ __forceinline__ void grid_barrier(DeviceState *st, unsigned &gen) {
    __syncthreads();
    ++gen;
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned target = gen * gridDim.x;
        if (atomicAdd(&st->bar_count, 1u) + 1u != target) {
            // bounded spin (a few seconds): a CTA that never arrives must not hang the device
            for (unsigned n = 0; ld_acquire(&st->bar_count) < target; ++n)
                if (n > (1u << 22)) { st->err_barrier = 1; break; }
        }
        __threadfence();
    }
    __syncthreads();
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
