// atom_lists.cu -- ATOM list mode: construction of the exact per-atom lists (cluster.cuh has the
// layout, atom_pairs.cu the kernels that walk them).
//
// Paper, "List filtering": a group's neighbour list is filtered down to "a list of
// atoms which really belong to a group's neighborhood", padded with phantom atoms.  Here the
// filtering is carried down to the single atom: every entry of an atom's list is a pair with
// R^2 <= r_c^2 for the positions of the build, so the pair kernels contain no cutoff test.  The
// candidates of an atom are the entries of its 8-atom cluster's list (cluster_build.cu).
//
// Pass 1 (k_atom_scan): one CTA per group, one warp per block, one lane per atom; chunk by chunk the
// staged positions are put in shared memory and every lane walks its cluster's list.  A hit is classified
//   FAR   x = R^3 w_i w_j >= x0 (e^-x below FP32 resolution: the Thole term is dropped) and
//         R >= R_far (z = beta R inside the range of the far-field erfcx fit), or
//   NEAR  otherwise (full formula),
// and appended to its class of the open segment.  Pass 2 (k_atom_deal, one warp per block) then puts
// every class of every segment into its final order through a per-warp shared-memory IMAGE (the
// image is 16 KB per warp: inside pass 1 it would leave room for 7 warps per SM, and that pass is
// latency bound):
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

// One class (far or near) of one lane's image.  The 16 column counters of a lane are bytes in shared
// memory, cnt[column * 32] (a register array indexed per lane would cost a dozen instructions per
// access): k_atom_lists is bound by its instruction count.
struct Deal {
    uint8_t *cnt;      // this lane's counters: cnt[b * 32], b = 0..15
    int novf = 0;      // entries on the overflow stack (top rows of the image)
    __device__ __forceinline__ void clear() {
#pragma unroll
        for (int b = 0; b < 16; ++b) cnt[b * 32] = 0;
        novf = 0;
    }
};

// rows of column j that lie inside a list of `len` entries
__device__ __forceinline__ unsigned col_cap(unsigned j, unsigned len) { return (len + 15u - j) >> 4; }     // (0 for j >= len: j <= 15)

// Put one entry into the image: into its own column, or, when that column is full, onto the overflow
// stack that grows down from row `top` of the image (branch-free: this pass is bound by its instruction
// stream, and a probing loop runs as long as its slowest lane).  The stack has `ovf_cap` cells above
// the rows the class can use; an entry that finds it full probes the next columns (rare).
__device__ __forceinline__ void deal(Deal &d, uint16_t *img, int colcap, unsigned l16, unsigned off, unsigned bank,
                                     int top, int ovf_cap) {
    unsigned b = bank, r = d.cnt[b * 32];
    bool ok = r < (unsigned)colcap;
    if (!ok && d.novf >= ovf_cap) {
        do {
            b = (b + 1) & 15u;
            r = d.cnt[b * 32];
        } while (r >= (unsigned)colcap);
        ok = true;
    }
    const unsigned t = ok ? ((b - l16) & 15u) + 16u * r : (unsigned)(top - d.novf);
    img[t * 32] = (uint16_t)off;
    d.cnt[b * 32] = (uint8_t)(r + (ok ? 1u : 0u));
    d.novf += ok ? 0 : 1;
}

// the next hole of the image in column order (there is one: the class is padded to its longest lane)
__device__ __forceinline__ void to_hole(const Deal &d, uint16_t *img, unsigned l16, unsigned len, unsigned &hb, uint16_t v) {
    unsigned hr = d.cnt[hb * 32];
    while (hr >= col_cap((hb - l16) & 15u, len)) {
        ++hb;
        hr = d.cnt[hb * 32];
    }
    img[(((hb - l16) & 15u) + 16u * hr) * 32] = v;
    d.cnt[hb * 32] = (uint8_t)(hr + 1);
}

// Entries of over-full columns and of the overflow stack -> holes of under-full columns (per lane, no
// cross-lane traffic).  First into the PARTNER column (j + 8) mod 16: its steps want the same index
// class mod 8, so the quarter warp's LDS.128 stays conflict-free and only the half warp's LDS.64 takes
// a second wavefront; what is left goes into any hole (those steps may conflict with one other lane).
__device__ __forceinline__ void level(Deal &d, uint16_t *img, unsigned l16, unsigned len, int top, unsigned rec_shift) {
    // pass 1: partner columns
    for (unsigned b = 0; b < 16; ++b) {
        const unsigned j = (b - l16) & 15u, pb = (b + 8u) & 15u, pj = (pb - l16) & 15u;
        unsigned cb = d.cnt[b * 32], cp = d.cnt[pb * 32];
        const unsigned capb = col_cap(j, len), capp = col_cap(pj, len);
        while (cb > capb && cp < capp) {
            --cb;
            img[(pj + 16u * cp) * 32] = img[(j + 16u * cb) * 32];
            img[(j + 16u * cb) * 32] = 0xffffu;
            ++cp;
        }
        d.cnt[b * 32] = (uint8_t)cb;
        d.cnt[pb * 32] = (uint8_t)cp;
    }
    // pass 2: whatever is still over the edge, into the holes in column order
    unsigned hb = 0;
    for (unsigned b = 0; b < 16; ++b) {
        const unsigned j = (b - l16) & 15u;
        const unsigned cb = d.cnt[b * 32];
        for (unsigned r = col_cap(j, len); r < cb; ++r) to_hole(d, img, l16, len, hb, img[(j + 16u * r) * 32]);
    }
    // pass 3: the overflow stack, partner column first
    for (int i = 0; i < d.novf; ++i) {
        const uint16_t v = img[(top - i) * 32];
        img[(top - i) * 32] = 0xffffu;
        const unsigned pb = (((unsigned)v >> rec_shift) + 8u) & 15u, pj = (pb - l16) & 15u;
        const unsigned cp = d.cnt[pb * 32];
        if (cp < col_cap(pj, len)) {
            img[(pj + 16u * cp) * 32] = v;
            d.cnt[pb * 32] = (uint8_t)(cp + 1);
        } else {
            to_hole(d, img, l16, len, hb, v);
        }
    }
}

// ---- pass 1: scan.  One CTA per group, one warp per block, one lane per atom.  The kernel is bound by
// its instruction count, so the appends are branch-free: a hit is written (predicated) into a small
// per-lane queue in shared memory -- FAR hits into a 16-entry ring from which every lane writes its
// own 16-byte row (8 entries, arrival order; pass 2 permutes them in place) as soon as it has one,
// NEAR hits into a buffer that waits until the length of the far part of the segment is known.
constexpr int FQ = 32;                  // entries of a lane's far ring (the last 32 far hits: close_segment moves some of them)

template <typename real>
__global__ void __launch_bounds__(GT)
k_atom_scan(ClusterWs ws, const typename Vec4<real>::type *__restrict__ gpos,
            const typename Vec4<real>::type *__restrict__ stage_pos, real rc2, real far_c, real far_r2,
            int s_chunk, DeviceState *st) {
    using vec4 = typename Vec4<real>::type;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    vec4 *s_pos = reinterpret_cast<vec4 *>(smem_raw);          // [s_chunk] | per warp: near buffer [NEAR_CAP][32], far ring [FQ][32] (u16)

    const int g = blockIdx.x, t = threadIdx.x, lane = t & 31, w = t >> 5;
    const int b0 = ws.group_first[g], nb = ws.group_first[g + 1] - b0;
    const int count = ws.stage_count[g];
    const size_t gbase = (size_t)g * ws.s_cap;
    const int n_chunks = atom_chunks_of(count, s_chunk);
    const bool active = w < nb;
    const int blk = b0 + (active ? w : 0);
    int2 *__restrict__ seg = ws.aseg + (size_t)blk * NSEG_MAX;
    // padding entries point at the (first) dummy record after the largest chunk of THIS group
    const unsigned dummy = (unsigned)atom_dummy_index(count, n_chunks) * (unsigned)sizeof(vec4);
    if (n_chunks > NCH_MAX) {                      // uniform over the CTA
        if (t == 0) st->atom_bad = 1;
        if (active && lane == 0) seg[0] = seg[NSEG_MAX - 1] = make_int2((int)(0xffu << 24), (int)dummy);
        return;
    }
    const unsigned magic = ((1u << 20) + (unsigned)n_chunks - 1u) / (unsigned)n_chunks;   // e / n for e < 2^16
    const int slot = blk * BLOCK + lane;
    const vec4 pi = gpos[slot];
    const real vi = cbrt(pi.w * pi.w);
    const int oct = slot >> 3;
    const int L = active ? ws.oct_len[oct] : 0;
    const uint4 *__restrict__ ent8 = reinterpret_cast<const uint4 *>(ws.entries + (size_t)oct * ws.l_cap);  // 8 entries per load
    const int L8 = L >> 3;                                                                                   // L is a multiple of 8
    uint4 *__restrict__ rows = reinterpret_cast<uint4 *>(ws.alist + (size_t)blk * ws.a_cap * 32) + lane;    // row r of this lane: rows[r * 32]
    const int rows_cap = ws.a_cap >> 3;
    const int fcap = ws.far_cap;
    uint16_t *nbuf = reinterpret_cast<uint16_t *>(smem_raw + (size_t)(s_chunk + 1) * sizeof(vec4)) +
                     (size_t)w * (NEAR_CAP + FQ) * 32 + lane;                            // nbuf[k * 32]
    uint16_t *fq = nbuf + NEAR_CAP * 32;                                                 // fq[(k & 15) * 32]

    int row_cur = 0, nseg = 0;
    long long slots = 0, slots_far = 0;
    bool bad = false;
    int kf = 0, kn = 0;                  // far / near entries of this lane in the open segment
    int fw = 0;                          // far entries of this lane already written to its rows (multiple of 8)

    // this lane's far row fw / 8 of the open segment from the ring; entries from `valid` on are padding
    auto put_row = [&](int valid) {
        unsigned v[8];
        const uint16_t *q8 = fq + (fw & (FQ - 1)) * 32;          // fw is a multiple of 8: the row's entries are q8[h * 32]
        if (valid - fw >= 8) {                                   // (the usual call: a whole row is waiting)
#pragma unroll
            for (int h = 0; h < 8; ++h) v[h] = q8[h * 32];
        } else {
#pragma unroll
            for (int h = 0; h < 8; ++h) v[h] = fw + h < valid ? q8[h * 32] : dummy;
        }
        const int r = row_cur + (fw >> 3);
        if (r < rows_cap) rows[(size_t)r * 32] = make_uint4(v[0] | (v[1] << 16), v[2] | (v[3] << 16), v[4] | (v[5] << 16), v[6] | (v[7] << 16));
        fw += 8;
    };
    // closes the open segment: pads both classes to the longest lane, writes the near rows and the descriptor
    auto close_segment = [&](int c) {
        int nmax = kn;
        for (int o = 16; o > 0; o >>= 1) nmax = max(nmax, __shfl_xor_sync(0xffffffffu, nmax, o));
        // A lane with fewer NEAR entries than the longest lane would pad its near class with dummies;
        // it fills those slots with its own last FAR entries instead (the full formula is exact for
        // them too).  Lanes with few near neighbours are the ones with many far ones, so this shortens
        // the far class of the warp: config 2: 141.7 -> 130.7 far slots per atom, near slots all useful.
        {
            const int m = min(min(2 * ((nmax + 1) >> 1) - kn, kf), FQ / 2);
            for (int k = 0; k < m; ++k) nbuf[(kn + k) * 32] = fq[((kf - m + k) & (FQ - 1)) * 32];
            kn += m;
            kf -= m;
            fw = min(fw, kf & ~7);               // the row that holds my new last far entry is rewritten below
        }
        int fmax = kf;
        for (int o = 16; o > 0; o >>= 1) fmax = max(fmax, __shfl_xor_sync(0xffffffffu, fmax, o));
        if (fmax + nmax == 0) return;
        const int ncf = (fmax + 1) >> 1, ncn = (nmax + 1) >> 1;              // calls of 2 entries
        const int fr = (ncf + 3) >> 2, nr = (ncn + 3) >> 2;                  // rows of 4 calls
        if (row_cur + fr + nr > rows_cap || nseg >= NSEG_MAX - 1) {
            bad = true;                                                       // capacity: CLUSTER lists are used
        } else {
            while (fw < 8 * fr) put_row(kf);                                  // my last (partial) row, then padding rows
            uint4 *out = rows + (size_t)(row_cur + fr) * 32;
            for (int r = 0; r < nr; ++r, out += 32) {
                unsigned v[8];
#pragma unroll
                for (int h = 0; h < 8; ++h) v[h] = 8 * r + h < kn ? nbuf[(8 * r + h) * 32] : dummy;
                *out = make_uint4(v[0] | (v[1] << 16), v[2] | (v[3] << 16), v[4] | (v[5] << 16), v[6] | (v[7] << 16));
            }
            if (lane == 0) seg[nseg] = make_int2(row_cur | (c << 24), ncf | (ncn << 16));
            ++nseg;
            row_cur += fr + nr;
            slots += 2 * (ncf + ncn);
            slots_far += 2 * ncf;
        }
        kf = 0; kn = 0; fw = 0;
    };

    // the walk over my cluster's list for chunk c; ONE: the group has a single chunk (the usual case:
    // entry = local index, no division by the chunk count and no membership test)
    auto walk_chunk = [&](int c, auto one_tag) {
        constexpr bool ONE = decltype(one_tag)::value;
        uint4 nxt = L8 > 0 ? ent8[0] : make_uint4(0, 0, 0, 0);
        bool open = true;                                // per lane: its cluster's list has entries left
        for (int v = 0; v < L8 && __any_sync(0xffffffffu, open); ++v) {
            const uint4 cur = nxt;
            if (v + 1 < L8) nxt = ent8[v + 1];           // one address per quarter warp, one load ahead
            const unsigned word[4] = {cur.x, cur.y, cur.z, cur.w};
            // the 8 entries of the vector are tested together (8 independent chains), then appended
            // without a branch: a predicated store into the ring / the near buffer and a counter
#pragma unroll
            for (int h = 0; h < 8; ++h) {
                const unsigned e = (word[h >> 1] >> ((h & 1) * 16)) & 0xffffu;
                const unsigned loc = ONE ? e : (e * magic) >> 20;              // e / n_chunks
                // padding entries are == count: ONE: they read the far record behind the chunk, no test needed
                bool hit = ONE || ((int)e < count && e - loc * (unsigned)n_chunks == (unsigned)c);
                if (h == 7) open = (int)e < count;                             // padding only at the end of a list
                const vec4 pj = s_pos[loc];                                    // (a padding entry reads one record past the chunk: inside the shared-memory block, and hit is false)
                const real Rx = pi.x - pj.x, Ry = pi.y - pj.y, Rz = pi.z - pj.z;
                const real r2 = Rx * Rx + Ry * Ry + Rz * Rz;
                hit = hit && r2 <= rc2 && r2 > (real)1e-10;
                const bool far = r2 * (vi * pj.w) >= far_c && r2 >= far_r2;     // x^(2/3) = R^2 (w_i w_j)^(2/3); far class off: both thresholds are -1
                const uint16_t off = (uint16_t)(loc * (unsigned)sizeof(vec4));
                if (hit && far) fq[(kf & (FQ - 1)) * 32] = off;
                if (hit && !far) nbuf[kn * 32] = off;
                kf += (hit && far) ? 1 : 0;
                kn += (hit && !far) ? 1 : 0;
            }
            if (kf - fw >= 8) put_row(kf);               // at most 15 entries were waiting: one row empties the ring enough
            // a vector adds at most 8 entries to a class: close the segment before pass 2's image or the
            // near buffer could overflow
            if (__any_sync(0xffffffffu, kf > fcap - 8 || kn > NEAR_CAP - 8)) close_segment(c);
        }
        close_segment(c);
    };
    for (int c = 0; c < n_chunks; ++c) {
        __syncthreads();
        for (int l = t, idx = c + t * n_chunks; idx < count; l += GT, idx += GT * n_chunks)
        {
            vec4 p = stage_pos[gbase + idx];
            p.w = cbrt(p.w * p.w);                       // the class test wants w^(2/3)
            s_pos[l] = p;
        }
        if (t == 0 && n_chunks == 1) {                   // the record the padding entries (== count) point at: far away
            vec4 far;
            far.x = far.y = far.z = (real)(-3.0f * PHANTOM_FAR); far.w = 0;
            s_pos[count] = far;
        }
        __syncthreads();
        if (!active) continue;
        if (n_chunks == 1) walk_chunk(c, TrueTag());
        else walk_chunk(c, FalseTag());
    }
    if (active && lane == 0) {
        seg[nseg] = seg[NSEG_MAX - 1] = make_int2(row_cur | (int)(0xffu << 24), (int)dummy);    // terminator (y = the dummy offset); total rows also in the last slot
        if (bad) st->atom_bad = 1;
        atomicAdd((unsigned long long *)&st->n_atom_entries, (unsigned long long)slots);
        atomicAdd((unsigned long long *)&st->n_atom_far, (unsigned long long)slots_far);
        atomicAdd((unsigned long long *)&st->n_atom_segments, (unsigned long long)nseg);
    }
}

// ---- pass 2: deal.  One warp per block: every class of every segment is read into the image in the
// bank-aware layout (header comment), levelled, and written back in place.
constexpr int DEAL_WARPS = 4;

__global__ void __launch_bounds__(DEAL_WARPS * 32)
k_atom_deal(ClusterWs ws, int n_blocks, int rec_bytes) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int blk = blockIdx.x * DEAL_WARPS + w;
    if (blk >= n_blocks) return;
    const int fcap = ws.far_cap;
    const int img_rows = fcap > NEAR_CAP ? fcap : NEAR_CAP;
    uint16_t *img = reinterpret_cast<uint16_t *>(smem_raw) + (size_t)w * img_rows * 32 + lane;       // img[row * 32]
    Deal D;
    D.cnt = smem_raw + (size_t)DEAL_WARPS * img_rows * 32 * sizeof(uint16_t) + (size_t)w * 512 + lane;
    const unsigned l16 = (unsigned)lane & 15u;
    uint4 *__restrict__ rows = reinterpret_cast<uint4 *>(ws.alist + (size_t)blk * ws.a_cap * 32) + lane;
    const int2 *__restrict__ seg = ws.aseg + (size_t)blk * NSEG_MAX;
    const unsigned dummy = (unsigned)seg[NSEG_MAX - 1].y;            // byte offset of the first dummy record
    const unsigned rec_shift = rec_bytes == 16 ? 4u : 5u;            // index class of an entry = (offset / record bytes) mod 16
    const unsigned n_loc = dummy / (unsigned)rec_bytes;
    for (int r = 0; r < img_rows; ++r) img[r * 32] = 0xffffu;
    D.clear();

    for (int d = 0; d < NSEG_MAX; ++d) {
        const int2 sd = seg[d];
        if (seg_chunk(sd) == 0xff) break;
        const int nc[2] = {seg_far_calls(sd), seg_near_calls(sd)};
        int r0 = seg_row0(sd);
        for (int cls = 0; cls < 2; ++cls) {
            const int nrow = (nc[cls] + 3) >> 2, len = 2 * nc[cls];
            uint4 *p = rows + (size_t)r0 * 32;
            r0 += nrow;
            if (nrow == 0 || 8 * nrow > img_rows) continue;          // (an over-long class keeps its arrival order)
            const int colcap = (8 * nrow + 15) >> 4;
            const int top = img_rows - 1;
            int ovf_cap = img_rows - 16 * colcap;                    // free rows above the cells the class can use
            if (ovf_cap < 0) ovf_cap = 0;
            uint4 nxt = p[0];
            for (int q = 0; q < nrow; ++q) {
                const uint4 e = nxt;
                if (q + 1 < nrow) nxt = p[(size_t)(q + 1) * 32];
                const unsigned v[8] = {e.x & 0xffffu, e.x >> 16, e.y & 0xffffu, e.y >> 16,
                                       e.z & 0xffffu, e.z >> 16, e.w & 0xffffu, e.w >> 16};
#pragma unroll
                for (int h = 0; h < 8; ++h)
                    if (v[h] < dummy) deal(D, img, colcap, l16, v[h], (v[h] >> rec_shift) & 15u, top, ovf_cap);      // (the scan pads with the first dummy)
            }
            level(D, img, l16, (unsigned)len, top, rec_shift);
            for (int q = 0; q < nrow; ++q) {
                unsigned v[8];
#pragma unroll
                for (int h = 0; h < 8; ++h) {
                    const int e = 8 * q + h;
                    const unsigned x = img[e * 32];
                    // padding: the dummy record of the index class this lane wants at this step
                    const unsigned pad = dummy + ((((unsigned)(e + lane) - n_loc) & 15u) << rec_shift);
                    v[h] = (e >= len || x == 0xffffu) ? pad : x;
                    img[e * 32] = 0xffffu;
                }
                p[(size_t)q * 32] = make_uint4(v[0] | (v[1] << 16), v[2] | (v[3] << 16), v[4] | (v[5] << 16), v[6] | (v[7] << 16));
            }
            // cells beyond the written rows that the spill of a full column touched
            for (int e = 8 * nrow; e < 16 * colcap && e < img_rows; ++e) img[e * 32] = 0xffffu;
            D.clear();
        }
    }
}

// ----------------------------------------------------------------------------- host side
static size_t deal_smem(const ClusterWs &ws) {
    const int img_rows = ws.far_cap > NEAR_CAP ? ws.far_cap : NEAR_CAP;
    return (size_t)DEAL_WARPS * ((size_t)img_rows * 32 * sizeof(uint16_t) + 512);
}

int atom_build(Ctx *c, cudaStream_t s) {
    ClusterWs ws = get_ws(c);
    const bool f64 = c->p.precision == TKHP_FP64;
    const int s_chunk = atom_chunk_capacity(f64, ws.chunk_cap);
    const size_t smem = (size_t)(s_chunk + 1) * (f64 ? sizeof(double4) : sizeof(float4)) + (size_t)GB * (NEAR_CAP + FQ) * 32 * sizeof(uint16_t);
    const double rc2 = c->p.cutoff * c->p.cutoff;
    // far class off (FP64, beta = 0): far_r2 < 0 puts every pair into the first class of rows, which
    // the kernels then evaluate with the full formula
    // a pair is FAR iff x = R^3 w_i w_j >= x0, tested as R^2 (w_i w_j)^(2/3) >= x0^(2/3), and R >= R_far
    const double x2 = c->far_on ? cbrt(c->far_x0 * c->far_x0) : -1.0, r2_far = c->far_on ? c->far_rmin * c->far_rmin : -1.0;
    if (f64)
        k_atom_scan<double><<<ws.n_groups, GT, smem, s>>>(ws, ws.gpos64, ws.stage_pos64, rc2, x2, r2_far, s_chunk, c->st);
    else
        k_atom_scan<float><<<ws.n_groups, GT, smem, s>>>(ws, ws.gpos32, ws.stage_pos32, (float)rc2, (float)x2,
                                                          (float)r2_far, s_chunk, c->st);
    k_atom_deal<<<div_up(c->n_blocks, DEAL_WARPS), DEAL_WARPS * 32, deal_smem(ws), s>>>(ws, c->n_blocks, f64 ? 32 : 16);
    c->n_launches += 2;
    TKHP_CUDA(c, cudaGetLastError());
    return TKHP_OK;
}

int atom_lists_configure(Ctx *c) {
    TKHP_CUDA(c, cudaFuncSetAttribute(k_atom_scan<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
    TKHP_CUDA(c, cudaFuncSetAttribute(k_atom_scan<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
    TKHP_CUDA(c, cudaFuncSetAttribute(k_atom_deal, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
    return TKHP_OK;
}

long long atom_slots(Ctx *c) { return 32LL * c->h_state->n_atom_entries; }

}  // namespace tkhp
