// atom_lists.cu -- ATOM list mode: construction of the exact per-atom lists (cluster.cuh has the
// layout, atom_pairs.cu the kernels that walk them).
//
// Paper, "List filtering": a group's neighbour list is filtered down to "a list of
// atoms which really belong to a group's neighborhood", padded with phantom atoms.  Here the
// filtering is carried down to the single atom: every entry of an atom's list is a pair with
// R^2 <= r_c^2 for the positions of the build, so the pair kernels contain no cutoff test.  The
// candidates of an atom are the entries of its 8-atom cluster's list (cluster_build.cu).
//
// One CTA per group, one warp per block, one lane per atom; chunk by chunk the staged positions
// are put in shared memory and every lane walks its cluster's list.  A hit is classified
//   FAR   x = R^3 w_i w_j >= x0 (e^-x below FP32 resolution: the Thole term is dropped) and
//         R >= R_far (z = beta R inside the range of the far-field erfcx fit), or
//   NEAR  otherwise (full formula),
// and dealt straight into its final position of a per-warp shared-memory IMAGE of the segment:
// the pair kernels gather a 16-byte and an 8-byte record from shared memory, one per lane and step;
// a quarter warp's LDS.128 (a half warp's LDS.64) is served in one wavefront only if its 8 (16)
// records have different indices mod 8 (mod 16).  Lane l therefore keeps 16 columns per class,
// column j = (index - l) mod 16 holding the rows j, j + 16, j + 32, ...: at step t lane l reads a
// record of index (t + l) mod 16 whenever it has one left.  When the chunk is exhausted (or the image is full) the warp pads the class to
// its longest lane (in calls of 2 entries), moves the entries of over-full columns into the holes
// of under-full ones (those steps may conflict), fills the remaining holes with the dummy record
// and writes the rows out, coalesced.  Order within a list only changes FP32 summation order.
#include "cluster.cuh"

namespace tkhp {

// one class (far or near) of one lane's image: 16 column counters of 8 bits
struct Deal {
    unsigned long long c0 = 0ull, c1 = 0ull;
    int k = 0;
    __device__ __forceinline__ unsigned get(unsigned b) const { return (unsigned)(((b & 8u) ? c1 : c0) >> (8 * (b & 7u))) & 0xffu; }
    __device__ __forceinline__ void inc(unsigned b) {
        const unsigned long long one = 1ull << (8 * (b & 7u));
        if (b & 8u) c1 += one; else c0 += one;
    }
};

// put one entry into the image; a full column spills into the next one (only a bank conflict later)
__device__ __forceinline__ void deal(Deal &d, uint16_t *img, int colcap, unsigned l16, unsigned off, unsigned bank) {
    unsigned b = bank, r = d.get(b);
    while (r >= (unsigned)colcap) {
        b = (b + 1) & 15u;
        r = d.get(b);
    }
    const unsigned t = ((b - l16) & 15u) + 16u * r;
    img[t * 32] = (uint16_t)off;
    d.inc(b);
    ++d.k;
}

// rows of column j that lie inside a list of `len` entries
__device__ __forceinline__ unsigned col_cap(unsigned j, unsigned len) { return j < len ? (len - j + 15u) >> 4 : 0u; }

// entries of over-full columns -> holes of under-full ones (per lane, no cross-lane traffic)
__device__ __forceinline__ void level(const Deal &d, uint16_t *img, unsigned l16, unsigned len) {
    unsigned hb = 0, hr = d.get(0);
    for (unsigned b = 0; b < 16; ++b) {
        const unsigned j = (b - l16) & 15u;
        const unsigned cb = d.get(b);
        for (unsigned r = col_cap(j, len); r < cb; ++r) {
            const uint16_t v = img[(j + 16u * r) * 32];
            while (hr >= col_cap((hb - l16) & 15u, len)) {
                ++hb;
                hr = d.get(hb);
            }
            img[(((hb - l16) & 15u) + 16u * hr) * 32] = v;
            ++hr;
        }
    }
}

template <typename real>
__global__ void __launch_bounds__(GT)
k_atom_lists(ClusterWs ws, const typename Vec4<real>::type *__restrict__ gpos,
             const typename Vec4<real>::type *__restrict__ stage_pos, real rc2, real far_x2, real far_r2,
             int s_chunk, DeviceState *st) {
    using vec4 = typename Vec4<real>::type;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    vec4 *s_pos = reinterpret_cast<vec4 *>(smem_raw);

    const int g = blockIdx.x, t = threadIdx.x, lane = t & 31, w = t >> 5;
    const int b0 = ws.group_first[g], nb = ws.group_first[g + 1] - b0;
    const int count = ws.stage_count[g];
    const size_t gbase = (size_t)g * ws.s_cap;
    const int n_chunks = atom_chunks_of(count, s_chunk);
    const bool active = w < nb;
    const int blk = b0 + (active ? w : 0);
    int2 *__restrict__ seg = ws.aseg + (size_t)blk * NSEG_MAX;
    if (n_chunks > NCH_MAX) {                      // uniform over the CTA
        if (t == 0) st->atom_bad = 1;
        if (active && lane == 0) seg[0] = seg[NSEG_MAX - 1] = make_int2((int)(0xffu << 24), 0);
        return;
    }
    const unsigned magic = ((1u << 20) + (unsigned)n_chunks - 1u) / (unsigned)n_chunks;   // e / n for e < 2^16
    const int slot = blk * BLOCK + lane;
    const vec4 pi = gpos[slot];
    const int oct = slot >> 3;
    const int L = active ? ws.oct_len[oct] : 0;
    const uint4 *__restrict__ ent8 = reinterpret_cast<const uint4 *>(ws.entries + (size_t)oct * ws.l_cap);  // 8 entries per load
    const int L8 = L >> 3;                                                                                   // L is a multiple of 8
    uint4 *__restrict__ rows = reinterpret_cast<uint4 *>(ws.alist + (size_t)blk * ws.a_cap * 32) + lane;    // row r of this lane: rows[r * 32]
    const int rows_cap = ws.a_cap >> 3;
    // padding entries point at the record after the largest chunk of THIS group (the kernels put a
    // far-away record with zero payload there)
    const unsigned dummy = (unsigned)atom_dummy_index(count, n_chunks) * (unsigned)sizeof(vec4);
    const unsigned l16 = (unsigned)lane & 15u;
    const int fcap = ws.far_cap, fcol = fcap >> 4, ncol = NEAR_CAP >> 4;
    uint16_t *img_f = reinterpret_cast<uint16_t *>(smem_raw + (size_t)s_chunk * sizeof(vec4)) +
                      (size_t)(active ? w : 0) * (fcap + NEAR_CAP) * 32 + lane;          // img[row * 32]
    uint16_t *img_n = img_f + (size_t)fcap * 32;

    int row_cur = 0, nseg = 0;
    long long slots = 0, slots_far = 0;
    bool bad = false;
    Deal F, N;
    if (active)
        for (int r = 0; r < fcap + NEAR_CAP; ++r) img_f[r * 32] = 0xffffu;

    // pads, levels and writes out the segment collected so far (warp-uniform control flow)
    auto flush = [&](int c) {
        int fmax = F.k, nmax = N.k;
        for (int o = 16; o > 0; o >>= 1) {
            fmax = max(fmax, __shfl_xor_sync(0xffffffffu, fmax, o));
            nmax = max(nmax, __shfl_xor_sync(0xffffffffu, nmax, o));
        }
        if (fmax + nmax == 0) return;
        const int ncf = (fmax + 1) >> 1, ncn = (nmax + 1) >> 1;              // calls of 2 entries
        const int fr = (ncf + 3) >> 2, nr = (ncn + 3) >> 2;                  // rows of 4 calls
        if (row_cur + fr + nr > rows_cap || nseg >= NSEG_MAX - 1) {
            bad = true;                                                       // capacity: CLUSTER lists are used
        } else {
            level(F, img_f, l16, 2u * ncf);
            level(N, img_n, l16, 2u * ncn);
            for (int part = 0; part < 2; ++part) {
                uint16_t *img = part ? img_n : img_f;
                const int nrow = part ? nr : fr, len = 2 * (part ? ncn : ncf);
                uint4 *out = rows + (size_t)(row_cur + (part ? fr : 0)) * 32;
                for (int q = 0; q < nrow; ++q, out += 32) {
                    unsigned v[8];
#pragma unroll
                    for (int h = 0; h < 8; ++h) {
                        const int e = 8 * q + h;
                        const unsigned x = img[e * 32];
                        v[h] = (e >= len || x == 0xffffu) ? dummy : x;
                        img[e * 32] = 0xffffu;
                    }
                    *out = make_uint4(v[0] | (v[1] << 16), v[2] | (v[3] << 16), v[4] | (v[5] << 16), v[6] | (v[7] << 16));
                }
                // rows of the image beyond the written ones that the spill of a full column touched
                const int used = part ? NEAR_CAP : fcap;
                for (int e = 8 * nrow; e < used; ++e) img[e * 32] = 0xffffu;
            }
            if (lane == 0) seg[nseg] = make_int2(row_cur | (c << 24), ncf | (ncn << 16));
            ++nseg;
            row_cur += fr + nr;
            slots += 2 * (ncf + ncn);
            slots_far += 2 * ncf;
        }
        F = Deal();
        N = Deal();
    };

    for (int c = 0; c < n_chunks; ++c) {
        __syncthreads();
        for (int l = t, idx = c + t * n_chunks; idx < count; l += GT, idx += GT * n_chunks)
            s_pos[l] = stage_pos[gbase + idx];
        __syncthreads();
        if (!active) continue;
        uint4 nxt = L8 > 0 ? ent8[0] : make_uint4(0, 0, 0, 0);
        bool open = true;                                // per lane: its cluster's list has entries left
        for (int v = 0; v < L8 && __any_sync(0xffffffffu, open); ++v) {
            const uint4 cur = nxt;
            if (v + 1 < L8) nxt = ent8[v + 1];           // one address per quarter warp, one load ahead
            const unsigned word[4] = {cur.x, cur.y, cur.z, cur.w};
            // the 8 entries of the vector are tested together (8 independent chains), then the hits
            // are dealt in list order
            unsigned loc[8];
            bool hit[8], far[8];
#pragma unroll
            for (int h = 0; h < 8; ++h) {
                const unsigned e = (word[h >> 1] >> ((h & 1) * 16)) & 0xffffu;
                loc[h] = (e * magic) >> 20;                        // e / n_chunks
                hit[h] = (int)e < count && e - loc[h] * (unsigned)n_chunks == (unsigned)c;   // padding entries are == count
                if (h == 7) open = (int)e < count;                 // padding only at the end of a list
            }
#pragma unroll
            for (int h = 0; h < 8; ++h) {
                const vec4 pj = s_pos[hit[h] ? loc[h] : 0u];
                const real Rx = pi.x - pj.x, Ry = pi.y - pj.y, Rz = pi.z - pj.z;
                const real r2 = Rx * Rx + Ry * Ry + Rz * Rz;
                const real ww = pi.w * pj.w;
                hit[h] = hit[h] && r2 <= rc2 && r2 > (real)1e-10;
                far[h] = ((r2 * r2 * r2) * (ww * ww) >= far_x2 && r2 >= far_r2) || far_r2 < (real)0;    // x^2 = R^6 (w_i w_j)^2
            }
#pragma unroll
            for (int h = 0; h < 8; ++h) {
                if (hit[h]) {
                    const unsigned off = loc[h] * (unsigned)sizeof(vec4);
                    if (far[h]) deal(F, img_f, fcol, l16, off, loc[h] & 15u);
                    else deal(N, img_n, ncol, l16, off, loc[h] & 15u);
                }
            }
            // a vector adds at most 8 entries to a class: start another segment before one overflows
            if (__any_sync(0xffffffffu, F.k > fcap - 8 || N.k > NEAR_CAP - 8)) flush(c);
        }
        flush(c);
    }
    if (active && lane == 0) {
        seg[nseg] = seg[NSEG_MAX - 1] = make_int2(row_cur | (int)(0xffu << 24), 0);    // terminator; total rows also in the last slot
        if (bad) st->atom_bad = 1;
        atomicAdd((unsigned long long *)&st->n_atom_entries, (unsigned long long)slots);
        atomicAdd((unsigned long long *)&st->n_atom_far, (unsigned long long)slots_far);
        atomicAdd((unsigned long long *)&st->n_atom_segments, (unsigned long long)nseg);
    }
}

// ----------------------------------------------------------------------------- host side
size_t atom_lists_smem(const ClusterWs &ws, bool f64, int nb_max) {
    const int s_chunk = atom_chunk_capacity(f64, ws.chunk_cap);
    return (size_t)s_chunk * (f64 ? sizeof(double4) : sizeof(float4)) +
           (size_t)nb_max * (ws.far_cap + NEAR_CAP) * 32 * sizeof(uint16_t);
}

int atom_build(Ctx *c, cudaStream_t s) {
    ClusterWs ws = get_ws(c);
    const bool f64 = c->p.precision == TKHP_FP64;
    const int s_chunk = atom_chunk_capacity(f64, ws.chunk_cap);
    const int nb_max = (c->n_blocks + ws.n_groups - 1) / ws.n_groups;
    const size_t smem = atom_lists_smem(ws, f64, nb_max);
    const double rc2 = c->p.cutoff * c->p.cutoff;
    // far class off (FP64, beta = 0): far_r2 < 0 puts every pair into the first class of rows, which
    // the kernels then evaluate with the full formula
    const double x2 = c->far_on ? c->far_x0 * c->far_x0 : 0.0, r2_far = c->far_on ? c->far_rmin * c->far_rmin : -1.0;
    if (f64)
        k_atom_lists<double><<<ws.n_groups, GT, smem, s>>>(ws, ws.gpos64, ws.stage_pos64, rc2, x2, r2_far, s_chunk, c->st);
    else
        k_atom_lists<float><<<ws.n_groups, GT, smem, s>>>(ws, ws.gpos32, ws.stage_pos32, (float)rc2, (float)x2,
                                                           (float)r2_far, s_chunk, c->st);
    c->n_launches += 1;
    TKHP_CUDA(c, cudaGetLastError());
    return TKHP_OK;
}

int atom_lists_configure(Ctx *c) {
    TKHP_CUDA(c, cudaFuncSetAttribute(k_atom_lists<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
    TKHP_CUDA(c, cudaFuncSetAttribute(k_atom_lists<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
    return TKHP_OK;
}

long long atom_slots(Ctx *c) { return 32LL * c->h_state->n_atom_entries; }

}  // namespace tkhp
