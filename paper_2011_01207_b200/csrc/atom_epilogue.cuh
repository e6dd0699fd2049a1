// atom_epilogue.cuh -- what every ATOM-mode T.mu kernel does once a lane holds (T p)_i: the parts of a
// shared block are added, the FP64 result is stored, and inside the PCG loop q and the block's share of
// p.q are formed (used by atom_pairs.cu and atom_stored.cu).
#pragma once
#include "cluster.cuh"
#include "reduce.cuh"

namespace tkhp {

static_assert(GT == RED_THREADS, "the fused PCG epilogue uses the 256-thread block reductions");

// PCG fusion (MODE_TMU): the lane that owns atom i holds (T p)_i when the
// list is exhausted, so q_i = p_i/alpha_i - (T p)_i - self p_i and the block's share of p.q are
// formed here instead of in a separate vector kernel.
struct PcgFuse {
    int on;
    double self;
    const double *vp;          // 3 n_pad, direction p (FP64)
    const double *inv_alpha;   // n_pad
    double *vq;                // 3 n_pad out
    double *part;              // 2 * n_groups block partials
};

// Common epilogue: add the parts of a block (part 1 first), store the FP64 result, and in the PCG
// loop form q = p/alpha - T p - self p and the block's share of p.q.
template <bool FUSE>
__device__ __forceinline__ void pair_epilogue(unsigned char *smem_raw, double dx, double dy, double dz, int wpb, int part,
                                              bool active, int slot, int n_pad, double *__restrict__ acc,
                                              DeviceState *st, const PcgFuse &fuse) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (wpb > 1) {                             // uniform over the CTA
        double *s_part = reinterpret_cast<double *>(smem_raw);         // [warp][xyz][lane], over the dead records
        __syncthreads();
        if (part > 0) {
            s_part[w * 96 + lane] = dx; s_part[w * 96 + 32 + lane] = dy; s_part[w * 96 + 64 + lane] = dz;
        }
        __syncthreads();
        if (part == 0)
            for (int k = 1; k < wpb; ++k) {
                dx += s_part[(w + k) * 96 + lane]; dy += s_part[(w + k) * 96 + 32 + lane]; dz += s_part[(w + k) * 96 + 64 + lane];
            }
    }
    const bool owner = active && part == 0;
    if (owner) {
        acc[slot] = dx;
        acc[n_pad + slot] = dy;
        acc[2 * (size_t)n_pad + slot] = dz;
    }
    if (FUSE && fuse.on) {
        double pq = 0, dummy = 0;
        if (owner) {
            const double ia = fuse.inv_alpha[slot];
            const double d[3] = {dx, dy, dz};
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const size_t o = (size_t)k * n_pad + slot;
                const double p = fuse.vp[o];
                const double q = p * ia - d[k] - fuse.self * p;
                fuse.vq[o] = q;
                pq += p * q;
            }
        }
        block_sum2(pq, dummy);
        if (grid_sum2_last_block(fuse.part, &st->ticket, pq, dummy) && threadIdx.x == 0) st->pq = pq;
    }
}

}  // namespace tkhp
