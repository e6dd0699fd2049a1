// cluster.cuh / cluster_build.cu / cluster_pairs.cu -- CLUSTER list mode: filtered cluster->atom lists with the neighbourhood of a
// group of blocks staged in shared memory.
//
// Paper, "List filtering": "By filtering every neighboring group, we can get a list
// of atoms which really belong to a group's neighborhood ... alpha in B_I if there is alpha_i in
// beta_I such that dist(alpha_i, alpha) <= d_cut + d_buff ... phantom atoms to complete the actual
// neighbor lists ... a loss of coalesced memory access pattern ... compensated by an increase of
// B_comp", +75% on their vdW kernel, then applied to "electrostatics and polarization".
//
// B200 redesign:
//  * the filter granularity is an 8-atom CLUSTER (a quarter warp), not the 32-atom block: with
//    r_c = 7 A a 32-atom block is as wide as the cutoff and only ~26% of (block atom, list atom)
//    slots are inside r_c; for 8-atom clusters it is ~49% (measured, DESIGN.md table 5.1);
//  * the filter radius is r_c (+0.01 A guard), not r_c + skin: the list is used for the positions
//    it was built from (one solve), the skin only enters the prescribed block-pair list;
//  * a CTA owns a GROUP of up to 8 consecutive blocks; every list atom of the group's clusters is
//    staged ONCE in shared memory (position already shifted into the group's frame, so no image
//    arithmetic in the pair loop), and list entries are 16-bit indices into that staging area:
//    the "loss of coalesced access" the paper notes becomes conflict-free LDS.128 (each quarter
//    warp reads one 16-byte record, broadcast to its 8 lanes);
//  * every lane owns one atom i and only ever updates atom i: no atomics, no j-side accumulator,
//    bit-reproducible results; FP32 partials are flushed into FP64 registers every 32 entries
//    (64-bit containers for accumulation);
//  * the number of groups is a whole multiple of (SM count x resident CTAs) whenever the system
//    is smaller than a few waves, so every SM gets the same number of blocks.
#pragma once
#include "common.cuh"
#include "pair_math.cuh"

namespace tkhp {

// compile-time flags handed to generic lambdas (one loop body, two instantiations, one uniform branch outside)
struct TrueTag { static constexpr bool value = true; };
struct FalseTag { static constexpr bool value = false; };

constexpr int GB = 8;                 // max blocks per group (= warps per CTA)
constexpr int GT = GB * 32;           // threads per CTA
constexpr int OCT = GB * 4;           // clusters per group
constexpr int CB_CAP = 1024;          // candidate blocks per group
constexpr int RESIDENT = 3;           // CTAs per SM the group count is rounded to
constexpr int B200_SMS = 148;
constexpr float GUARD = 0.01f;        // list radius = r_c + GUARD (FP32 build arithmetic is safe)
constexpr int NCH_MAX = 16;           // ATOM mode: max staging chunks per group
constexpr int NSEG_MAX = 2 * NCH_MAX; // ATOM mode: list segments (descriptors) per block, incl. the terminator
constexpr int NEAR_CAP = 48;          // ATOM mode builder: near entries per lane and segment (image rows)
constexpr int ATOM_SMEM = 56 * 1024;  // ATOM mode: shared memory of the T.mu kernel per CTA (4 CTAs / SM)

// ATOM mode chunking of a group's staged atoms.  The shared-memory chunk holds s_max records; a
// group with `count` staged atoms uses n = ceil(count / s_max) chunks, chunk c = the staged atoms
// with index == c (mod n), stored at local index idx / n.  Interleaving (instead of consecutive
// runs of the spatially ordered staging area) splits every atom's neighbours evenly over the
// chunks, so that padding each chunk's lists to the longest lane of the warp stays cheap.
__host__ __device__ inline int atom_chunk_capacity(bool f64, int user_cap) {
    const int fit = (ATOM_SMEM / (f64 ? 64 : 32) - 1) & ~31;     // records of pos + mu
    return (user_cap > 0 && user_cap < fit) ? user_cap : fit;
}
__host__ __device__ inline int atom_chunks_of(int count, int s_chunk) {
    return count < 1 ? 1 : (count + s_chunk - 1) / s_chunk;
}
// Padding entries point at DUMMY records (far away, zero payload) that follow the group's largest
// chunk: N_DUMMY of them, one per index class mod 16, so that a padding entry can be given the class
// its lane wants at that step (atom_lists.cu: no bank conflict with the lanes that read real records).
constexpr int N_DUMMY = 16;
// local index of the first dummy record of a group: one past its largest chunk (<= s_chunk)
__host__ __device__ inline int atom_dummy_index(int count, int n_chunks) {
    return count < 1 ? 0 : (count + n_chunks - 1) / n_chunks;
}

// Rows of the far image the list builder keeps per warp (atom_lists.cu): 1.25 x the expected number
// of neighbours of an atom in one chunk + 24, so that a chunk normally needs one segment (an
// under-estimate only costs padding: the builder starts another segment when the image is full).
inline int atom_far_cap(const tkhp_params *p, int n_blocks, int n_groups, bool f64) {
    double per_chunk = 96.0;
    if (p->box > 0.0) {
        const double rho = p->n_atoms / (p->box * p->box * p->box);
        const double nb = 4.18879 * p->cutoff * p->cutoff * p->cutoff * rho;
        // staged atoms of a typical group: its atoms fill a (somewhat elongated) cube, widened by r_c
        const double atoms = (double)BLOCK * n_blocks / n_groups;
        double edge = 1.25 * cbrt(atoms / rho) + 2.0 * p->cutoff;
        if (edge > p->box) edge = p->box;
        const double staged = 0.45 * rho * edge * edge * edge;     // a low estimate: fewer chunks, larger image
        const int chunk = atom_chunk_capacity(f64, p->max_stage_per_chunk);
        const int n_chunks = (int)(staged / chunk) + 1;
        per_chunk = nb / n_chunks;
    }
    int cap = ((int)(1.25 * per_chunk) + 24 + 15) & ~15;
    if (cap < 32) cap = 32;
    if (cap > 224) cap = 224;           // 16 KB of image per warp
    return cap;
}

struct ClusterWs {
    int n_groups, s_cap, l_cap;
    int32_t *group_first;             // n_groups + 1
    float4 *gpos32;                   // n_pad: atom in its group's frame (x,y,z,w)
    double4 *gpos64;
    int32_t *stage_count;             // n_groups
    int32_t *stage_atom;              // n_groups * s_cap: sorted slot of each staged atom
    float4 *stage_pos32;              // n_groups * s_cap: position in the group's frame (+w)
    double4 *stage_pos64;
    uint32_t *stage_mask;             // n_groups * s_cap: which clusters of the group list the atom
    uint16_t *entries;                // (n_pad/8) * l_cap
    int32_t *oct_len;                 // n_pad/8: padded list length (equal within a warp)
    // ATOM list mode (atom_lists.cu, atom_pairs.cu): per-atom lists, one u16 BYTE OFFSET into the
    // staged chunk per entry (record index * 16 in MIXED, * 32 in FP64), laid out per block as ROWS
    // [row][lane][8 entries]: 16 bytes per lane, one coalesced 512-byte row per warp.  A block's
    // rows are a sequence of SEGMENTS, each described by one int2 of `aseg`:
    //   x = first row | chunk << 24,   y = far calls | near calls << 16   (a call = 2 entries)
    // the FAR rows (pairs whose Thole damping has died out and whose z = beta R lies in the range
    // of the far-field fit: no Thole term, 2 MUFU) come first, the NEAR rows follow on the next row
    // boundary; both are padded to the longest lane of the warp in units of one call.  A chunk
    // normally has one segment; the builder starts another when its shared-memory image is full.
    // The sequence ends with a terminator (chunk 0xff, x & 0xffffff = total rows of the block), which
    // is repeated in the last slot of the block's descriptors.
    int chunk_cap;                    // tkhp_params.max_stage_per_chunk (0 = automatic)
    int a_cap;                        // entries per lane and block (multiple of 8)
    int far_cap;                      // builder image: far entries per lane and segment (multiple of 16)
    uint16_t *alist;                  // n_blocks * a_cap * 32
    int2 *aseg;                       // n_blocks * NSEG_MAX
};

__host__ __device__ __forceinline__ int seg_chunk(int2 d) { return (int)((unsigned)d.x >> 24); }
__host__ __device__ __forceinline__ int seg_row0(int2 d) { return d.x & 0xffffff; }
__host__ __device__ __forceinline__ int seg_far_calls(int2 d) { return d.y & 0xffff; }
__host__ __device__ __forceinline__ int seg_near_calls(int2 d) { return (int)((unsigned)d.y >> 16); }

inline int choose_groups(int n_blocks) {
    const int base = (n_blocks + GB - 1) / GB;
    const int wave = B200_SMS * RESIDENT;
    if (base >= 4 * wave) return base;
    int g = ((base + wave - 1) / wave) * wave;
    if (g > n_blocks) g = n_blocks;
    return g;
}

inline void size_caps(const tkhp_params *p, int n_blocks, int *s_cap, int *l_cap) {
    const long long n_pad = (long long)n_blocks * BLOCK;
    long long s, l;
    if (p->box > 0.0) {
        const double rho = p->n_atoms / (p->box * p->box * p->box);
        const double e = 1.3 * cbrt(GT / rho);
        double edge = e + 2.0 * (p->cutoff + 1.0);
        if (edge > p->box) edge = p->box;
        s = (long long)(1.25 * edge * edge * edge * rho) + 64;
        const double r = p->cutoff + 3.0;
        l = (long long)(1.5 * 4.18879 * r * r * r * rho) + 64;
    } else {
        s = 8192;
        l = 2048;
    }
    if (p->max_nbrs_per_cluster > 0) l = p->max_nbrs_per_cluster;
    if (s > n_pad + 1) s = n_pad + 1;
    if (l > n_pad + 8) l = n_pad + 8;
    if (s > 65535) s = 65535;          // 16-bit entries
    *s_cap = (int)((s + 63) & ~63LL);
    *l_cap = (int)((l + 7) & ~7LL);
}

inline size_t carve_cluster(const tkhp_params *p, int n_blocks, void *base, ClusterWs *out) {
    Carver w(base);
    ClusterWs ws;
    const size_t n_pad = (size_t)n_blocks * BLOCK;
    ws.n_groups = choose_groups(n_blocks);
    size_caps(p, n_blocks, &ws.s_cap, &ws.l_cap);
    const bool f64 = p->precision == TKHP_FP64;
    const size_t gs = (size_t)ws.n_groups * ws.s_cap;
    ws.group_first = w.take<int32_t>(ws.n_groups + 1);
    ws.gpos32 = w.take<float4>(n_pad);
    ws.gpos64 = f64 ? w.take<double4>(n_pad) : nullptr;
    ws.stage_count = w.take<int32_t>(ws.n_groups);
    ws.stage_atom = w.take<int32_t>(gs);
    ws.stage_pos32 = w.take<float4>(gs);
    ws.stage_pos64 = f64 ? w.take<double4>(gs) : nullptr;
    ws.stage_mask = w.take<uint32_t>(gs);
    ws.entries = w.take<uint16_t>((n_pad / CLUSTER) * ws.l_cap);
    ws.oct_len = w.take<int32_t>(n_pad / CLUSTER);
    ws.a_cap = 0; ws.far_cap = 0; ws.alist = nullptr; ws.aseg = nullptr;
    ws.chunk_cap = p->max_stage_per_chunk;
    if (p->list_mode == TKHP_LIST_ATOM) {
        long long a;
        if (p->max_nbrs_per_atom > 0) {
            a = p->max_nbrs_per_atom;
        } else if (p->box > 0.0) {
            const double rho = p->n_atoms / (p->box * p->box * p->box);
            const double r = p->cutoff + 0.05;
            a = (long long)(1.6 * 4.18879 * r * r * r * rho) + 112;
        } else {
            a = 1024;
        }
        if (a > (long long)n_pad + 16 * NCH_MAX) a = (long long)n_pad + 16 * NCH_MAX;
        ws.a_cap = (int)((a + 7) & ~7LL);
        ws.far_cap = atom_far_cap(p, n_blocks, ws.n_groups, f64);
        ws.alist = w.take<uint16_t>((size_t)n_blocks * ws.a_cap * 32);
        ws.aseg = w.take<int2>((size_t)n_blocks * NSEG_MAX);
    }
    w.take<char>(256);
    if (out) *out = ws;
    return w.off;
}


inline ClusterWs get_ws(Ctx *c) {
    ClusterWs ws;
    carve_cluster(&c->p, c->n_blocks, c->cl_ws, &ws);
    return ws;
}

}  // namespace tkhp
