// a1 — neighbour search: periodic / open cell list -> CSR pair list (§2.2.2).
//
// Atoms are binned into cells of edge >= rc(1+2^-20) and counting-sorted by cell (ties broken by the
// caller's index, so the internal order is deterministic).  One block per cell stages its <= 27 stencil
// cells in shared memory as centre-relative fp32 coordinates and tests every (centre, candidate) pair
// in fp32; pairs within the fp32 error margin of a cutoff are decided by the canonical fp64 predicate of
// include/dhp.h, so the list is bit-exact.  Kept pairs go to a fixed-stride
// temporary row; a second pass assigns CSR offsets and orders each row by (angular first, then
// radial-only) x neighbour species.  Rows hold sorted-slot indices.  Rows of the AEV / MLP buffers are
// grouped by the central atom's species (stable in sorted order), each group starting at a multiple
// of ROW_ALIGN rows so that one MLP tile (and one CTA pair of two tiles) never mixes networks.
#include <algorithm>
#include <string.h>

#include "dhp_internal.cuh"

namespace dhp {

// ---------------------------------------------------------------------------------------------
// helpers
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned f2ord(float f) {
    unsigned u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float ord2f(unsigned u) {
    return __uint_as_float((u & 0x80000000u) ? (u & 0x7fffffffu) : ~u);
}

// exclusive scan of n ints by ONE block of 1024 threads; out[n] = total.  Every thread takes 8 consecutive elements,
// so 8192 elements go through one round of warp / block scans (the 6 859 cells of the 98 k box: one round)
__device__ void block_scan_excl(const int* __restrict__ in, int* __restrict__ out, int n) {
    constexpr int IPT = 8;
    __shared__ int warp_sums[32];
    __shared__ int carry_s;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) carry_s = 0;
    __syncthreads();
    for (int base = 0; base < n; base += 1024 * IPT) {
        const int i0 = base + tid * IPT;
        int v[IPT];
        int sum = 0;
#pragma unroll
        for (int i = 0; i < IPT; ++i) { v[i] = i0 + i < n ? in[i0 + i] : 0; sum += v[i]; }
        int x = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) warp_sums[wid] = x;
        __syncthreads();
        if (wid == 0) {
            int w = warp_sums[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                int y = __shfl_up_sync(0xffffffffu, w, o);
                if (lane >= o) w += y;
            }
            warp_sums[lane] = w;
        }
        __syncthreads();
        const int carry = carry_s;
        int run = carry + (wid ? warp_sums[wid - 1] : 0) + x - sum;
#pragma unroll
        for (int i = 0; i < IPT; ++i) {
            if (i0 + i < n) out[i0 + i] = run;
            run += v[i];
        }
        __syncthreads();
        if (tid == 1023) carry_s = carry + warp_sums[31];
        __syncthreads();
    }
    if (tid == 0) out[n] = carry_s;
}

// Verlet-skin reuse (dhp_set_skin): whether a call rebuilds the cell grid and the candidate list or reuses them is
// decided ON THE DEVICE (k_reuse_check), so the host enqueues both paths and every kernel of the path not taken
// returns at once.  gate == nullptr (skin off): no check.
#define DHP_GATE(gate, want) do { if ((gate) != nullptr && *(gate) != (want)) return; } while (0)

// ---------------------------------------------------------------------------------------------
// grid setup
// ---------------------------------------------------------------------------------------------
__global__ void k_bbox(const float* __restrict__ pos, int n, unsigned* __restrict__ bbox, const int* __restrict__ gate) {
    DHP_GATE(gate, 1);
    float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f};
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x)
        for (int c = 0; c < 3; ++c) {
            float v = pos[3 * i + c];
            lo[c] = fminf(lo[c], v);
            hi[c] = fmaxf(hi[c], v);
        }
    for (int c = 0; c < 3; ++c) {
        for (int o = 16; o; o >>= 1) {
            lo[c] = fminf(lo[c], __shfl_xor_sync(0xffffffffu, lo[c], o));
            hi[c] = fmaxf(hi[c], __shfl_xor_sync(0xffffffffu, hi[c], o));
        }
        if ((threadIdx.x & 31) == 0) {
            atomicMin(&bbox[c], f2ord(lo[c]));
            atomicMax(&bbox[3 + c], f2ord(hi[c]));
        }
    }
}

__global__ void k_setup_grid(Grid* g, int periodic, double Lx, double Ly, double Lz, double rc,
                             const unsigned* __restrict__ bbox, int max_cells, int by_molecule, int n_mol,
                             const int* __restrict__ gate, int* __restrict__ rebuild_count, int* __restrict__ cand_bad) {
    DHP_GATE(gate, 1);
    if (threadIdx.x || blockIdx.x) return;
    if (rebuild_count) ++*rebuild_count;
    *cand_bad = 0;                                           // a full build starts a fresh candidate list
    const double edge = rc * (1.0 + 9.5367431640625e-07);   // rc (1 + 2^-20): binning slack
    double L[3] = {Lx, Ly, Lz};
    g->periodic = periodic;
    g->by_molecule = by_molecule;
    if (by_molecule) {
        for (int c = 0; c < 3; ++c) {
            g->L[c] = 0; g->origin[c] = 0; g->inv_cell[c] = 0; g->nc[c] = 1;
            g->edge[c] = 0; g->inv_L[c] = 0; g->wrap[c] = 0; g->Lf[c] = 0.f; g->inv_Lf[c] = 0.f;
        }
        g->nc[0] = n_mol;
        g->ncell = n_mol;
        return;
    }
    double ext[3];
    for (int c = 0; c < 3; ++c) {
        if (periodic) {
            g->L[c] = L[c];
            g->origin[c] = 0.0;
            ext[c] = L[c];
            g->nc[c] = max(1, (int)floor(L[c] / edge));
        } else {
            double lo = (double)ord2f(bbox[c]), hi = (double)ord2f(bbox[3 + c]);
            g->L[c] = 0.0;
            g->origin[c] = lo;
            ext[c] = fmax(hi - lo, 0.0) * (1.0 + 1e-9) + 1e-6;   // max coordinate maps below nc
            g->nc[c] = max(1, (int)floor(ext[c] / edge));
        }
    }
    // bounded workspace: fewer, larger cells if the box is huge and dilute (still correct)
    while ((double)g->nc[0] * g->nc[1] * g->nc[2] > (double)max_cells) {
        int big = 0;
        if (g->nc[1] > g->nc[big]) big = 1;
        if (g->nc[2] > g->nc[big]) big = 2;
        g->nc[big] = max(1, g->nc[big] / 2);
    }
    for (int c = 0; c < 3; ++c) {
        g->inv_cell[c] = (double)g->nc[c] / ext[c];
        g->edge[c] = ext[c] / (double)g->nc[c];
        g->inv_L[c] = periodic ? 1.0 / L[c] : 0.0;
        g->wrap[c] = (periodic && g->nc[c] < 3) ? 1 : 0;
        g->Lf[c] = (float)L[c];
        g->inv_Lf[c] = periodic ? (float)(1.0 / L[c]) : 0.f;
    }
    g->ncell = g->nc[0] * g->nc[1] * g->nc[2];
}

__device__ __forceinline__ int cell_coord(double x, double L, double origin, double inv_cell, int nc, int periodic) {
    double t;
    if (periodic) {
        double f = x / L;
        f -= floor(f);
        t = f * (double)nc;
    } else {
        t = (x - origin) * inv_cell;
    }
    int c = (int)t;
    return min(max(c, 0), nc - 1);
}

__global__ void k_assign_cells(const float* __restrict__ pos, const int* __restrict__ species, int n,
                               const int* __restrict__ mol_offsets, int n_mol, const Grid* __restrict__ g,
                               int* __restrict__ cell_of, int* __restrict__ cell_count, int* __restrict__ status,
                               const int* __restrict__ gate) {
    DHP_GATE(gate, 1);
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int s = species[i];
    if (s < 0 || s >= NSP) atomicCAS(status, 0, DHP_E_SPECIES);   // never over a CAPACITY fault: k_scan_blocks derives cand_bad from the word
    int cell;
    if (g->by_molecule) {
        int lo = 0, hi = n_mol;            // largest m with mol_offsets[m] <= i
        while (hi - lo > 1) {
            int mid = (lo + hi) >> 1;
            if (mol_offsets[mid] <= i) lo = mid; else hi = mid;
        }
        cell = lo;
    } else {
        int c[3];
        for (int d = 0; d < 3; ++d)
            c[d] = cell_coord((double)pos[3 * i + d], g->L[d], g->origin[d], g->inv_cell[d], g->nc[d], g->periodic);
        cell = c[0] + g->nc[0] * (c[1] + g->nc[1] * c[2]);
    }
    cell_of[i] = cell;
    atomicAdd(&cell_count[cell], 1);
}

__global__ void k_scan_cells(const int* __restrict__ cnt, int* __restrict__ start, const Grid* __restrict__ g,
                             const int* __restrict__ gate) {
    DHP_GATE(gate, 1);
    block_scan_excl(cnt, start, g->ncell);
}

__global__ void k_scatter(const int* __restrict__ cell_of, int n, const int* __restrict__ cell_start,
                          int* __restrict__ cell_fill, int* __restrict__ perm, const int* __restrict__ gate) {
    DHP_GATE(gate, 1);
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int c = cell_of[i];
    perm[cell_start[c] + atomicAdd(&cell_fill[c], 1)] = i;
}

// one warp per cell: order its atoms by caller index (deterministic internal order), then gather
__global__ void k_sort_gather(const float* __restrict__ pos, const int* __restrict__ species,
                              const Grid* __restrict__ g, const int* __restrict__ cell_start, const int* __restrict__ perm_in,
                              int* __restrict__ perm, int* __restrict__ inv_perm, float4* __restrict__ spos,
                              int* __restrict__ smol, const uint8_t* __restrict__ central, unsigned char* __restrict__ snc,
                              const int* __restrict__ gate, float* __restrict__ pos_ref) {
    DHP_GATE(gate, 1);
    const int c = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (c >= g->ncell) return;
    const int b = cell_start[c], e = cell_start[c + 1];
    for (int a = b + lane; a < e; a += 32) {
        const int v = perm_in[a];
        int rank = 0;
        for (int q = b; q < e; ++q) rank += perm_in[q] < v;     // caller indices are distinct
        const int dst = b + rank;
        perm[dst] = v;
        inv_perm[v] = dst;
        int s = species[v];
        s = min(max(s, 0), NSP - 1);
        spos[dst] = make_float4(pos[3 * v], pos[3 * v + 1], pos[3 * v + 2], __int_as_float(s));
        smol[dst] = g->by_molecule ? c : 0;
        if (central) snc[dst] = central[v] ? 0 : 1;
        if (pos_ref) { pos_ref[3 * v] = pos[3 * v]; pos_ref[3 * v + 1] = pos[3 * v + 1]; pos_ref[3 * v + 2] = pos[3 * v + 2]; }
    }
}

// ---------------------------------------------------------------------------------------------
// species-grouped rows, ordered inside a species group by the feature blocks the atom can touch
//
// One 128-row MLP tile runs one network, so rows are grouped by the central atom's species (groups start at
// multiples of ROW_TILE).  G1 / B1 skip the 64-wide feature blocks that are zero for a whole tile, so inside a
// group rows are ordered by a class derived from the atom's own block mask: the highest angular block it can
// touch (blocks are ordered common species first, dhp_internal.cuh) and whether it sees a rare species radially.
// Atoms with nested neighbour-species sets (water-only < near the solute < near a sulfur ...) then share tiles
// and the tile masks stay small.  The order is deterministic (stable in sorted-slot order inside a class).
// ---------------------------------------------------------------------------------------------
constexpr int RB = 256;           // slots per block in the row assignment
constexpr int NCLS = 32;          // classes per species
constexpr int NKEY = NSP * NCLS;  // 224 row keys

__device__ __forceinline__ int row_key(int s, unsigned m) {
    const unsigned ang = m & 0x3fffu;
    const int hi = ang ? 32 - __clz(ang) : 0;                 // 0 (no angular block) .. 14
    return s * NCLS + 2 * hi + (int)((m >> 15) & 1u);
}

// blk_hist is key-major: blk_hist[key * nrb + block]
__global__ void __launch_bounds__(RB)
k_rowkey_hist(const float4* __restrict__ spos, const unsigned* __restrict__ amask, const unsigned char* __restrict__ snc, int n, int nrb,
              int* __restrict__ blk_hist, const int* __restrict__ gate) {
    DHP_GATE(gate, 1);
    __shared__ int h[NKEY];
    for (int k = threadIdx.x; k < NKEY; k += RB) h[k] = 0;
    __syncthreads();
    const int a = blockIdx.x * RB + threadIdx.x;
    if (a < n && !(snc && snc[a])) atomicAdd(&h[row_key(__float_as_int(spos[a].w), amask[a])], 1);   // non-central atoms get no row
    __syncthreads();
    for (int k = threadIdx.x; k < NKEY; k += RB) blk_hist[(size_t)k * nrb + blockIdx.x] = h[k];
}

// single block of 1024 threads, warps take keys round-robin: exclusive scan over blocks per key, then the key starts
// (species groups aligned to ROW_ALIGN)
// one block per species, one warp per class key: exclusive scan of the key's counts over the row blocks; the block that
// finishes last (ticket counter, zeroed with the per-call arena) turns the species totals into the group starts
__global__ void __launch_bounds__(1024)
k_rowkey_scan(int* __restrict__ blk_hist, int nrb, int* __restrict__ sp_count, int* __restrict__ sp_start, int* __restrict__ key_start,
              int* __restrict__ done, const int* __restrict__ gate) {
    DHP_GATE(gate, 1);
    __shared__ int tot[NCLS];
    __shared__ int last_s;
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int s = blockIdx.x;
    {
        const int key = s * NCLS + w;
        int* hk = blk_hist + (size_t)key * nrb;
        int run = 0;
        constexpr int CH = 16;                              // 16 x 32 counts are requested at once: one memory latency per
        for (int base = 0; base < nrb; base += 32 * CH) {   // 512 blocks of a key instead of one per 32
            int v[CH];
#pragma unroll
            for (int c = 0; c < CH; ++c) { const int bb = base + 32 * c + lane; v[c] = bb < nrb ? hk[bb] : 0; }
#pragma unroll
            for (int c = 0; c < CH; ++c) {
                if (base + 32 * c >= nrb) break;
                const int bb = base + 32 * c + lane;
                int x = v[c];
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    int y = __shfl_up_sync(0xffffffffu, x, o);
                    if (lane >= o) x += y;
                }
                if (bb < nrb) hk[bb] = run + x - v[c];
                run += __shfl_sync(0xffffffffu, x, 31);
            }
        }
        if (lane == 0) tot[w] = run;
    }
    __syncthreads();
    if (w == 0) {                                          // lane = class: offsets of the keys inside the species group
        const int c = tot[lane];
        int x = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        key_start[s * NCLS + lane] = x - c;
        if (lane == 31) sp_count[s] = x;
        __threadfence();                                   // every lane's writes are device-visible before the ticket is taken
        __syncwarp();
        if (lane == 31) last_s = atomicAdd(done, 1) == NSP - 1;
    }
    __syncthreads();
    if (!last_s) return;
    __threadfence();
    __shared__ int starts[NSP + 1];
    if (threadIdx.x == 0) {
        int start = 0;
        for (int q = 0; q < NSP; ++q) {
            starts[q] = start;
            sp_start[q] = start;
            const int c = ((volatile int*)sp_count)[q];
            start += (c + ROW_ALIGN - 1) / ROW_ALIGN * ROW_ALIGN;
        }
        starts[NSP] = start;
        sp_start[NSP] = start;
        sp_count[NSP] = 0;
    }
    __syncthreads();
    if (threadIdx.x < NKEY) key_start[threadIdx.x] = ((volatile int*)key_start)[threadIdx.x] + starts[threadIdx.x / NCLS];
}

__global__ void __launch_bounds__(RB)
k_rowkey_rank(const float4* __restrict__ spos, const unsigned* __restrict__ amask, const unsigned char* __restrict__ snc, int n, int nrb,
              const int* __restrict__ blk_hist,
              const int* __restrict__ key_start, int* __restrict__ rowmap, int* __restrict__ row_species,
              int* __restrict__ row_slot, unsigned* __restrict__ tile_mask, const int* __restrict__ gate) {
    DHP_GATE(gate, 1);
    __shared__ int wcnt[RB / 32][NKEY];
    for (int k = threadIdx.x; k < (RB / 32) * NKEY; k += RB) (&wcnt[0][0])[k] = 0;
    __syncthreads();
    const int a = blockIdx.x * RB + threadIdx.x;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int s = 0, key = -1;
    unsigned m = 0;
    if (a < n && !(snc && snc[a])) { s = __float_as_int(spos[a].w); m = amask[a]; key = row_key(s, m); }
    const unsigned grp = __match_any_sync(0xffffffffu, key);
    const int rank_in_warp = __popc(grp & ((1u << lane) - 1u));
    if (key >= 0 && rank_in_warp == 0) wcnt[w][key] = __popc(grp);
    __syncthreads();
    if (a >= n) return;
    if (key < 0) { rowmap[a] = -1; return; }
    int before = 0;
    for (int q = 0; q < w; ++q) before += wcnt[q][key];
    const int row = key_start[key] + blk_hist[(size_t)key * nrb + blockIdx.x] + before + rank_in_warp;
    rowmap[a] = row;
    row_species[row] = s;
    row_slot[row] = a;
    // tile masks, kept equal within a tile pair (ROW_ALIGN): the lanes of the warp that fall into the same pair combine
    // their masks first, one lane per pair does the atomics
    const int pair = row / ROW_ALIGN;
    const unsigned act = __activemask();
    const unsigned grp2 = __match_any_sync(act, pair);
    const unsigned mm = __reduce_or_sync(grp2, m);
    if (mm && lane == __ffs(grp2) - 1) {
        atomicOr(&tile_mask[2 * pair], mm);
        atomicOr(&tile_mask[2 * pair + 1], mm);
    }
}

// ---------------------------------------------------------------------------------------------
// pass 1: one block per cell; the <= 27 stencil cells are staged in shared memory as fp32 coordinates
// relative to the centre cell (minimum image applied in fp64 at staging), so the inner loop is plain
// fp32.  A pair whose fp32 R^2 lies within a proven margin of rcr^2 or rca^2 is decided by the
// canonical fp64 predicate on the ORIGINAL coordinates; every other pair is decided by fp32 alone
// (its fp32 error is smaller than its distance to the threshold), so the list is still bit-exact.
// ---------------------------------------------------------------------------------------------
struct Stencil {
    int n[3];
    int c[3][3];
};

__device__ __forceinline__ void make_stencil(const Grid& g, int cell, Stencil& st) {
    if (g.by_molecule) {
        st.n[0] = st.n[1] = st.n[2] = 1;
        st.c[0][0] = cell; st.c[1][0] = 0; st.c[2][0] = 0;
        return;
    }
    int cc[3] = {cell % g.nc[0], (cell / g.nc[0]) % g.nc[1], cell / (g.nc[0] * g.nc[1])};
    for (int d = 0; d < 3; ++d) {
        int nc = g.nc[d], k = 0;
        if (g.periodic) {
            if (nc >= 3) {
                st.c[d][k++] = (cc[d] + nc - 1) % nc;
                st.c[d][k++] = cc[d];
                st.c[d][k++] = (cc[d] + 1) % nc;
            } else {                      // 1 or 2 cells on this axis: every cell once (Q19)
                for (int q = 0; q < nc; ++q) st.c[d][k++] = q;
            }
        } else {
            for (int q = cc[d] - 1; q <= cc[d] + 1; ++q)
                if (q >= 0 && q < nc) st.c[d][k++] = q;
        }
        st.n[d] = k;
    }
}

// The canonical predicate: fp64, no FMA contraction, d -= L*rint(d/L).
__device__ __forceinline__ double pair_r2(const float4& pi, const float4& pj, const Grid& g) {
    double d[3] = {(double)pj.x - (double)pi.x, (double)pj.y - (double)pi.y, (double)pj.z - (double)pi.z};
    if (g.periodic) {
#pragma unroll
        for (int c = 0; c < 3; ++c) d[c] = __dsub_rn(d[c], __dmul_rn(g.L[c], rint(__ddiv_rn(d[c], g.L[c]))));
    }
    return __dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2]));
}

// predicated 4-byte global store (keeps the hot loop of k_pairs free of branches)
__device__ __forceinline__ void st_if(bool p, unsigned* a, unsigned v) {
    asm volatile("{ .reg .pred q; setp.ne.u32 q, %0, 0; @q st.global.u32 [%1], %2; }" ::"r"((unsigned)p), "l"(a), "r"(v) : "memory");
}

constexpr int P1_THREADS = 128;
constexpr int ROWS_PER_BLK = 64;        // granularity of the block-sum scan that yields the CSR offsets
constexpr int CAND_TILE = 1024;        // candidates staged per tile (16 KB)
constexpr unsigned ENT_RADIAL_ONLY = 0x80000000u;   // temp-row entry: bit 31 = beyond rca, bits 28..30 = species, low 28 = slot

template <bool WRAP, bool SKIN>
__global__ void __launch_bounds__(P1_THREADS, 8)
k_pairs(const float4* __restrict__ spos, const Grid* __restrict__ gp, const int* __restrict__ cell_start, double rcr2,
        double rca2, int stride, int* __restrict__ cnt, unsigned* __restrict__ tmp, int* __restrict__ blk_sum,
        int* __restrict__ status, const unsigned char* __restrict__ snc, const int* __restrict__ gate, float rs2f,
        int cstride, int* __restrict__ cand_cnt, unsigned* __restrict__ cand_out) {
    DHP_GATE(gate, 1);
    __shared__ Grid g;
    __shared__ float4 cand[CAND_TILE + 32];
    __shared__ int seg_cell_b[28], seg_off[28], nseg_s;
    __shared__ float bmax_s[P1_THREADS / 32];
    if (threadIdx.x == 0) g = *gp;
    __syncthreads();
    const int cell = blockIdx.x;
    if (cell >= g.ncell) return;
    const int cb = cell_start[cell], ce = cell_start[cell + 1];
    if (ce == cb) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (snc) {
        // partial evaluation (one rank's slab of central atoms): a cell without a central atom needs no candidates at
        // all - its rows are empty.  7/8 of the cells at world size 8.
        bool any = false;
        for (int i = cb + (int)threadIdx.x; i < ce; i += P1_THREADS) any |= snc[i] == 0;
        if (!__syncthreads_or(any)) {
            for (int i = cb + (int)threadIdx.x; i < ce; i += P1_THREADS) { cnt[i] = 0; if (SKIN) cand_cnt[i] = 0; }
            return;
        }
    }

    // candidate segments: one per non-empty stencil cell (warp 0: lane <-> stencil cell, ballot-compacted)
    if (warp == 0) {
        Stencil st;
        make_stencil(g, cell, st);
        const int nst = st.n[0] * st.n[1] * st.n[2];
        int b = 0, cntc = 0;
        if (lane < nst) {
            const int ix = lane % st.n[0], iy = (lane / st.n[0]) % st.n[1], iz = lane / (st.n[0] * st.n[1]);
            const int c = g.by_molecule ? st.c[0][0] : st.c[0][ix] + g.nc[0] * (st.c[1][iy] + g.nc[1] * st.c[2][iz]);
            b = cell_start[c];
            cntc = cell_start[c + 1] - b;
        }
        int x = cntc;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        const unsigned m = __ballot_sync(0xffffffffu, cntc > 0);
        const int slot = __popc(m & ((1u << lane) - 1u));
        if (cntc > 0) { seg_cell_b[slot] = b; seg_off[slot] = x - cntc; }
        if (lane == 31) { const int ns = __popc(m); seg_cell_b[ns] = 0; seg_off[ns] = x; nseg_s = ns; }
    }
    __syncthreads();
    const int nseg = nseg_s;
    const int ncand = seg_off[nseg];

    // centre of the block's cell (reference point of the relative coordinates)
    double ctr[3];
    if (g.by_molecule) {
        const float4 p0 = spos[cb];
        ctr[0] = p0.x; ctr[1] = p0.y; ctr[2] = p0.z;
    } else {
        int cc[3] = {cell % g.nc[0], (cell / g.nc[0]) % g.nc[1], cell / (g.nc[0] * g.nc[1])};
#pragma unroll
        for (int d = 0; d < 3; ++d) ctr[d] = g.origin[d] + ((double)cc[d] + 0.5) * g.edge[d];
    }
    const bool wrapx = g.wrap[0], wrapy = g.wrap[1], wrapz = g.wrap[2];
    const float Lx = g.Lf[0], Ly = g.Lf[1], Lz = g.Lf[2];
    const float iLx = g.inv_Lf[0], iLy = g.inv_Lf[1], iLz = g.inv_Lf[2];
    const float rcr2f = (float)rcr2, rca2f = (float)rca2;
    const float rcr = sqrtf(rcr2f), rca = sqrtf(rca2f);
    const unsigned lt = (1u << lane) - 1u;

    for (int t0 = 0; t0 < ncand; t0 += CAND_TILE) {
        const int tn = min(CAND_TILE, ncand - t0);
        // ---- stage the tile -------------------------------------------------------------------
        float bmax = 0.f;
        int sg = 0;                                    // f only grows along a thread's walk: so does its segment
        for (int t = threadIdx.x; t < tn; t += P1_THREADS) {
            const int f = t0 + t;
            while (sg + 1 < nseg && seg_off[sg + 1] <= f) ++sg;
            const int j = seg_cell_b[sg] + (f - seg_off[sg]);
            const float4 pj = spos[j];
            double r[3] = {(double)pj.x - ctr[0], (double)pj.y - ctr[1], (double)pj.z - ctr[2]};
            if (g.periodic) {
#pragma unroll
                for (int d = 0; d < 3; ++d) r[d] -= g.L[d] * rint(r[d] * g.inv_L[d]);
            }
            const float x = (float)r[0], y = (float)r[1], z = (float)r[2];
            bmax = fmaxf(bmax, fmaxf(fabsf(x), fmaxf(fabsf(y), fabsf(z))));
            cand[t] = make_float4(x, y, z, __int_as_float(j | (__float_as_int(pj.w) << 28)));
        }
        if (threadIdx.x < 32) cand[tn + threadIdx.x] = make_float4(1.0e15f, 1.0e15f, 1.0e15f, __int_as_float(0x0fffffff));
        for (int o = 16; o; o >>= 1) bmax = fmaxf(bmax, __shfl_xor_sync(0xffffffffu, bmax, o));
        if (lane == 0) bmax_s[warp] = bmax;
        __syncthreads();
        float B = 0.f;
#pragma unroll
        for (int q = 0; q < P1_THREADS / 32; ++q) B = fmaxf(B, bmax_s[q]);
        // fp32 error bound of R^2 near a cutoff rc: |err| <= rc B 2^-19 + rc^2 2^-22; doubled
        const float mr = rcr * B * 3.8146973e-06f + rcr2f * 4.7683716e-07f;
        const float ma = rca * B * 3.8146973e-06f + rca2f * 4.7683716e-07f;
        // candidates of the Verlet-skin list: everything the fp32 test cannot exclude from R <= rcr + skin
        const float rs2_incl = SKIN ? rs2f + (sqrtf(rs2f) * B * 3.8146973e-06f + rs2f * 4.7683716e-07f) : 0.f;

        // ---- centre atoms of this cell, one warp each ----------------------------------------
        for (int i = cb + warp; i < ce; i += P1_THREADS / 32) {
            if (snc && snc[i]) {               // not a central atom of this call: an empty row
                if (lane == 0 && t0 == 0) { cnt[i] = 0; if (SKIN) cand_cnt[i] = 0; }
                continue;
            }
            // the centre's own relative coordinates: same arithmetic as the staged copy
            const float4 pio = spos[i];
            double ri[3] = {(double)pio.x - ctr[0], (double)pio.y - ctr[1], (double)pio.z - ctr[2]};
            if (g.periodic) {
#pragma unroll
                for (int d = 0; d < 3; ++d) ri[d] -= g.L[d] * rint(ri[d] * g.inv_L[d]);
            }
            const float pix = (float)ri[0], piy = (float)ri[1], piz = (float)ri[2];
            const int base0 = t0 ? cnt[i] : 0;
            const int cbase0 = (SKIN && t0) ? cand_cnt[i] : 0;
            int base = base0, cbase = cbase0;
            unsigned* trow = tmp + (size_t)i * stride;
            unsigned* crow = SKIN ? cand_out + (size_t)i * cstride : nullptr;
            asm volatile("" : "+l"(trow), "+l"(crow));      // keep the row pointers in registers
            // fast pass: fp32 alone decides and only remembers whether any candidate fell inside a margin; such a row
            // (about one in 2000) is then redone by the exact pass, which overwrites the same entries
            // distance of R^2 to either threshold, minimum over the candidates (self and dummies included: harmless)
            float near_r = 1.0e30f, near_a = 1.0e30f;
            {
                const float4* cp = cand + lane;
                int lin = lane;
#pragma unroll 4
                for (int c0 = 0; c0 < tn; c0 += 32, cp += 32, lin += 32) {      // warp-uniform trip count (ballots inside)
                    const float4 c = *cp;                  // the tile is padded with far-away dummies
                    const unsigned jj = __float_as_uint(c.w);
                    float dx = c.x - pix, dy = c.y - piy, dz = c.z - piz;
                    if (WRAP) {
                        if (wrapx) dx -= Lx * rintf(dx * iLx);
                        if (wrapy) dy -= Ly * rintf(dy * iLy);
                        if (wrapz) dz -= Lz * rintf(dz * iLz);
                    }
                    const float r2 = dx * dx + dy * dy + dz * dz;
                    const bool other = (jj & 0x0fffffffu) != (unsigned)i && (!WRAP || lin < tn);
                    const float ur = rcr2f - r2, ua = rca2f - r2;       // sign bit of ua: beyond the angular cutoff
                    const bool in_r = other & (ur >= 0.f);
                    near_r = fminf(near_r, fabsf(ur));
                    near_a = fminf(near_a, fabsf(ua));
                    const unsigned m = __ballot_sync(0xffffffffu, in_r);
                    const unsigned pos = (unsigned)base + __popc(m & lt);
                    st_if(in_r & (pos < (unsigned)stride), trow + pos, jj | (__float_as_uint(ua) & ENT_RADIAL_ONLY));
                    base += __popc(m);
                    if (SKIN) {
                        const bool in_c = other & (r2 <= rs2_incl);
                        const unsigned mc = __ballot_sync(0xffffffffu, in_c);
                        const unsigned cpos = (unsigned)cbase + __popc(mc & lt);
                        st_if(in_c & (cpos < (unsigned)cstride), crow + cpos, jj);
                        cbase += __popc(mc);
                    }
                }
            }
            const bool amb_seen = near_r <= mr || near_a <= ma;
            if (__any_sync(0xffffffffu, amb_seen)) {
                base = base0;
                for (int c0 = 0; c0 < tn; c0 += 32) {
                    const float4 c = cand[c0 + lane];
                    const int jj = __float_as_int(c.w);
                    float dx = c.x - pix, dy = c.y - piy, dz = c.z - piz;
                    if (WRAP) {
                        if (wrapx) dx -= Lx * rintf(dx * iLx);
                        if (wrapy) dy -= Ly * rintf(dy * iLy);
                        if (wrapz) dz -= Lz * rintf(dz * iLz);
                    }
                    const float r2 = dx * dx + dy * dy + dz * dz;
                    const bool other = (jj & 0x0fffffff) != i && (!WRAP || c0 + lane < tn);
                    bool in_r = other && r2 <= rcr2f;
                    bool in_a = other && r2 <= rca2f;
                    if (other && (fabsf(r2 - rcr2f) <= mr || fabsf(r2 - rca2f) <= ma)) {
                        const double r2d = pair_r2(pio, spos[jj & 0x0fffffff], g);
                        in_r = r2d <= rcr2;
                        in_a = r2d <= rca2;
                    }
                    const unsigned m = __ballot_sync(0xffffffffu, in_r);
                    const int pos = base + __popc(m & lt);
                    if (in_r && pos < stride) trow[pos] = (unsigned)jj | (in_a ? 0u : ENT_RADIAL_ONLY);
                    base += __popc(m);
                }
            }
            if (lane == 0) {
                if (SKIN) {
                    if (cbase > cstride) { atomicExch(status, DHP_E_CAPACITY); cbase = cstride; }
                    cand_cnt[i] = cbase;
                }
                if (base > stride) { atomicExch(status, DHP_E_CAPACITY); base = stride; }
                cnt[i] = base;
                if (t0 + CAND_TILE >= ncand) atomicAdd(&blk_sum[i / ROWS_PER_BLK], base);
            }
        }
        __syncthreads();
    }
}

// exclusive scan of the per-256-atom block sums; total > pair_cap empties the list (status CAPACITY)
// A capacity fault of this call (a truncated temporary or candidate row in k_pairs / k_refilter, or the overflow above)
// also marks the candidate list as unusable (cand_bad): the next call with list reuse then rebuilds instead of
// filtering a truncated candidate list (k_reuse_check reads the flag, a full build clears it).
__global__ void k_scan_blocks(const int* __restrict__ blk_sum, int* __restrict__ blk_off, int nblk, int64_t pair_cap,
                              int* __restrict__ status, int* __restrict__ cand_bad) {
    block_scan_excl(blk_sum, blk_off, nblk);
    __syncthreads();
    if (threadIdx.x == 0) {
        const int ovf = (blk_off[nblk] < 0 || (int64_t)blk_off[nblk] > pair_cap) ? 1 : 0;
        if (ovf) atomicExch(status, DHP_E_CAPACITY);
        blk_off[nblk + 1] = ovf;
        if (*(volatile int*)status == DHP_E_CAPACITY) *cand_bad = 1;
    }
}

constexpr int MAX_STRIDE_CHUNKS = 6;    // tmp_stride <= 192

// one row of the pair list, by one warp: the ni unordered entries at src (pass-1 format) are ordered by (angular first,
// then radial-only) x neighbour species into col[row_start ..), the 14 run lengths, the angular count and the
// feature-block mask of the atom are stored; with reuse_rows the tile mask of the atom's (kept) row is refreshed too.
// sg: 16 ints of shared memory private to the warp.
// species of the two members of internal pair `lane` (lo | hi << 4): depends on the lane only, so callers compute it once
__device__ __forceinline__ int lane_pair_species(int lane) {
    if (lane >= NPAIR) return 0;
    int hi = 0;
    while ((hi + 1) * (hi + 2) / 2 <= lane) ++hi;
    return prio_sp(lane - hi * (hi + 1) / 2) | (prio_sp(hi) << 4);
}

__device__ __forceinline__ void order_row(const unsigned* __restrict__ src, int ni, int row_start, int i, int lane, int lane_pair, int* sg,
                                          int* __restrict__ col, int* __restrict__ n_ang, unsigned short* __restrict__ seg_cnt,
                                          unsigned* __restrict__ amask, bool reuse_rows, const int* __restrict__ rowmap,
                                          unsigned* __restrict__ tile_mask) {
    const unsigned lt = (1u << lane) - 1u;
    unsigned e[MAX_STRIDE_CHUNKS];
#pragma unroll
    for (int k = 0; k < MAX_STRIDE_CHUNKS; ++k) e[k] = (k * 32 + lane < ni) ? src[k * 32 + lane] : 0xffffffffu;
    if (lane < 16) sg[lane] = 0;
    __syncwarp();
    // counts per key = class * 8 + species (class 0: angular, 1: radial-only); 15 = no entry
#pragma unroll
    for (int k = 0; k < MAX_STRIDE_CHUNKS; ++k) {
        if (k * 32 < ni) {
            const int key = (e[k] == 0xffffffffu) ? 15 : (int)((e[k] >> 28) & 15u);
            const unsigned m = __match_any_sync(0xffffffffu, key);
            if ((m & lt) == 0) sg[key] += __popc(m);      // group leader; keys are distinct across leaders
            __syncwarp();
        }
    }
    // lane k < 16 owns key k: exclusive prefix over keys -> segment starts
    int cnt_k = lane < 16 ? sg[lane] : 0;
    if (lane == 15 || lane == 7) cnt_k = 0;
    {   // which 64-wide feature blocks of this row's AEV can be non-zero (internal column order, dhp_internal.cuh)
        const unsigned has1 = __ballot_sync(0xffffffffu, cnt_k > 0), has2 = __ballot_sync(0xffffffffu, cnt_k > 1);
        const unsigned am = has1 & 0x7fu, am2 = has2 & 0x7fu, rm = (am | (has1 >> 8)) & 0x7fu;
        bool pp = false;
        if (lane < NPAIR) {                                   // lane = internal pair index
            const int sa = lane_pair & 15, sb = lane_pair >> 4;
            pp = (sa == sb) ? ((am2 >> sa) & 1u) != 0 : (((am >> sa) & (am >> sb)) & 1u) != 0;
        }
        const unsigned pm = __ballot_sync(0xffffffffu, pp);
        const bool bb = lane < 14 ? ((pm >> (2 * lane)) & 3u) != 0 : lane == 14 ? (rm & 0x0fu) != 0 : lane == 15 ? (rm & 0x70u) != 0 : false;
        const unsigned bmask = __ballot_sync(0xffffffffu, bb);
        if (lane == 0) {
            amask[i] = bmask;
            if (reuse_rows && bmask) {
                const int row = rowmap[i];
                if (row >= 0) { atomicOr(&tile_mask[(row / ROW_TILE) & ~1], bmask); atomicOr(&tile_mask[(row / ROW_TILE) | 1], bmask); }
            }
        }
    }
    int x = cnt_k;
#pragma unroll
    for (int o = 1; o < 16; o <<= 1) {
        int y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
    }
    const int na = __shfl_sync(0xffffffffu, x, 7);
    if (lane < 16) {
        int v = cnt_k;
        if (lane == 7) v = na;
        if (lane == 15) v = ni - na;
        seg_cnt[(size_t)i * 16 + lane] = (unsigned short)v;
    }
    if (lane == 0) n_ang[i] = na;
    __syncwarp();
    if (lane < 16) sg[lane] = row_start + x - cnt_k;
    __syncwarp();
#pragma unroll
    for (int k = 0; k < MAX_STRIDE_CHUNKS; ++k) {
        if (k * 32 < ni) {
            const int key = (e[k] == 0xffffffffu) ? 15 : (int)((e[k] >> 28) & 15u);
            const unsigned m = __match_any_sync(0xffffffffu, key);
            const int base = sg[key];
            if (key != 15) col[base + __popc(m & lt)] = (int)(e[k] & 0x0fffffffu);
            __syncwarp();
            if ((m & lt) == 0) sg[key] = base + __popc(m);
            __syncwarp();
        }
    }

}

// pass 2: ROWS_PER_BLK atoms per block; rows get their CSR offsets, entries are ordered by (angular first, then
// radial-only) x neighbour species, and the 14 segment sizes of every row are stored for the AEV kernels.
constexpr int P2_THREADS = 256;

__global__ void __launch_bounds__(P2_THREADS)
k_rows(const unsigned* __restrict__ tmp, int stride, const int* __restrict__ cnt, const int* __restrict__ blk_off, int nblk,
       int n, int* __restrict__ row_ptr, int* __restrict__ col, int* __restrict__ n_rad, int* __restrict__ n_ang,
       unsigned short* __restrict__ seg_cnt, unsigned* __restrict__ amask, const int* __restrict__ gate,
       const int* __restrict__ rowmap, unsigned* __restrict__ tile_mask) {
    __shared__ int wsum[ROWS_PER_BLK / 32];
    __shared__ int rstart[ROWS_PER_BLK];
    __shared__ int rcnt[ROWS_PER_BLK];
    // list reuse: the row assignment of the last full build stays, the tile masks follow the current feature-block masks
    const bool reuse_rows = gate != nullptr && *gate == 0;
    __shared__ int segs[P2_THREADS / 32][16];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int i0 = blockIdx.x * ROWS_PER_BLK;
    const bool ovf = blk_off[nblk + 1] != 0;
    if (tid < ROWS_PER_BLK) {
        const int a = i0 + tid;
        const int c = (a < n && !ovf) ? cnt[a] : 0;
        int x = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) wsum[warp] = x;
        rstart[tid] = x - c;
    }
    __syncthreads();
    if (tid < ROWS_PER_BLK) {
        const int a = i0 + tid;
        int before = ovf ? 0 : blk_off[blockIdx.x];
        for (int q = 0; q < warp; ++q) before += wsum[q];
        const int start = before + rstart[tid];
        const int c = (a < n && !ovf) ? cnt[a] : 0;
        if (a < n) { row_ptr[a] = start; n_rad[a] = c; }
        if (a == n - 1) row_ptr[n] = start + c;
        rstart[tid] = start;
        rcnt[tid] = c;
    }
    __syncthreads();

    int* sg = segs[warp];
    const int lane_pair = lane_pair_species(lane);
    for (int q = warp; q < ROWS_PER_BLK; q += P2_THREADS / 32) {
        const int i = i0 + q;
        if (i >= n) break;
        order_row(tmp + (size_t)i * stride, rcnt[q], rstart[q], i, lane, lane_pair, sg, col, n_ang, seg_cnt, amask, reuse_rows, rowmap, tile_mask);
    }
}

// ---------------------------------------------------------------------------------------------
// Verlet-skin reuse ("atomic positions do not move much between two time-steps").
// The full build records every pair within rcr + skin (candidates).  While no atom has moved more than skin / 2
// from the positions of that build, every pair within rcr now is a candidate, so the exact list of this call is
// the candidates filtered by the canonical predicate on the CURRENT positions: still bit-exact.  The cell grid,
// the sorted order, the species-grouped row assignment and the candidate rows are reused; pairs, rows' internal
// order, feature-block masks and tile masks are recomputed.
// ---------------------------------------------------------------------------------------------
__global__ void k_set_flag(int* flag, int v) { *flag = v; }

// flag := 1 (rebuild) if any atom moved more than skin/2 (thr2 = (skin/2)^2, shaved so that fp32 rounding errs on
// the safe side), changed species, or changed its central / non-central role
__global__ void k_reuse_check(const float* __restrict__ pos, const int* __restrict__ species, const float* __restrict__ pos_ref,
                              const float4* __restrict__ spos, const int* __restrict__ inv_perm, const uint8_t* __restrict__ central,
                              const unsigned char* __restrict__ snc, int n, float thr2, int* __restrict__ flag,
                              const int* __restrict__ cand_bad, const int* __restrict__ mol_offsets, const int* __restrict__ smol) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool bad = i == 0 && *cand_bad != 0;                     // the candidate list was truncated by a capacity fault
    if (i < n) {
        const float dx = pos[3 * i] - pos_ref[3 * i], dy = pos[3 * i + 1] - pos_ref[3 * i + 1], dz = pos[3 * i + 2] - pos_ref[3 * i + 2];
        const float d2 = dx * dx + dy * dy + dz * dz;
        const int slot = inv_perm[i];
        bad = !(d2 <= thr2) || species[i] != __float_as_int(spos[slot].w);      // NaN positions also force a rebuild
        if (central) bad |= (central[i] ? 0 : 1) != snc[slot];
        // the molecule table is identified by its address on the host side; its CONTENTS are checked here: atom i must
        // still lie in the molecule it was binned into
        if (mol_offsets) { const int m = smol[slot]; bad |= !(mol_offsets[m] <= i && i < mol_offsets[m + 1]); }
    }
    if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) *flag = 1;
}

__global__ void k_reset_rows(int* __restrict__ row_slot, int* __restrict__ row_species, int max_rows, const int* __restrict__ gate) {
    DHP_GATE(gate, 1);
    for (int r = blockIdx.x * blockDim.x + threadIdx.x; r < max_rows; r += gridDim.x * blockDim.x) { row_slot[r] = -1; row_species[r] = -1; }
}

// reuse: current positions into the sorted copy (species bits stay)
__global__ void k_regather(const float* __restrict__ pos, const int* __restrict__ perm, int n, float4* __restrict__ spos,
                           const int* __restrict__ gate) {
    DHP_GATE(gate, 0);
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= n) return;
    const int v = perm[a];
    spos[a] = make_float4(pos[3 * v], pos[3 * v + 1], pos[3 * v + 2], spos[a].w);
}

// reuse: one warp per central atom filters its candidates in fp32.  The inputs are fp32, so pj - pi in fp32 is the
// correctly rounded exact difference (relative error 2^-24); the minimum-image shift by the fp32 box edge (exact: the
// box IS fp32) adds at most 2 * 2^-24 dm, dm = the largest raw coordinate difference of the pair, so a component is
// off by <= 3 * 2^-24 dm.  Pairs whose fp32 R^2 lies within the resulting margin of a cutoff are decided by the
// canonical fp64 predicate, all others by fp32 alone: the list stays bit-exact.
constexpr int RF_WARPS = 4;
constexpr int RF_UNROLL = 4;
struct BoxArg { double L[3]; float Lf[3], iLf[3]; int periodic; };
__device__ __forceinline__ double pair_r2_box(const float4& pi, const float4& pj, const BoxArg& bx) {
    double d[3] = {(double)pj.x - (double)pi.x, (double)pj.y - (double)pi.y, (double)pj.z - (double)pi.z};
    if (bx.periodic) {
#pragma unroll
        for (int c = 0; c < 3; ++c) d[c] = __dsub_rn(d[c], __dmul_rn(bx.L[c], rint(__ddiv_rn(d[c], bx.L[c]))));
    }
    return __dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2]));
}

__global__ void __launch_bounds__(RF_WARPS * 32)
k_refilter(const float4* __restrict__ spos, const __grid_constant__ BoxArg bx, const unsigned* __restrict__ cand,
           const int* __restrict__ cand_cnt, int cstride, double rcr2, double rca2, int stride, int n, int* __restrict__ cnt,
           unsigned* __restrict__ tmp, int* __restrict__ blk_sum, int* __restrict__ status, const unsigned char* __restrict__ snc,
           const int* __restrict__ gate) {
    const int lane = threadIdx.x & 31;
    const int i = blockIdx.x * RF_WARPS + (threadIdx.x >> 5);
    if (i >= n) return;
    // everything the warp needs first is requested at once (the candidate row's address does not depend on its
    // length), so a warp pays two dependent memory latencies - this batch, then the gathers - not five
    const unsigned* row = cand + (size_t)i * cstride;
    unsigned e[RF_UNROLL];
#pragma unroll
    for (int u = 0; u < RF_UNROLL; ++u) e[u] = (32 * u + lane < cstride) ? row[32 * u + lane] : 0u;
    const int gv = *gate;
    const int nc = cand_cnt[i];
    const float4 pi = spos[i];
    const bool skip = snc != nullptr && snc[i] != 0;
    if (gv != 0) return;                                      // this call rebuilds: nothing to do here
    if (skip) { if (lane == 0) cnt[i] = 0; return; }
    const bool per = bx.periodic != 0;
    const float Lx = bx.Lf[0], Ly = bx.Lf[1], Lz = bx.Lf[2], iLx = bx.iLf[0], iLy = bx.iLf[1], iLz = bx.iLf[2];
    const float rcr2f = (float)rcr2, rca2f = (float)rca2;
    const float rcr = sqrtf(rcr2f), rca = sqrtf(rca2f);
    // margin of a pair: |err(R^2)| <= 2 sqrt(3) R (3 * 2^-24 dm) + 3 * 2^-24 R^2 with dm its largest raw coordinate difference; doubled
    const float kr = 2.0f * 2.0f * rcr * 3.0f * 5.9604645e-08f, ka = 2.0f * 2.0f * rca * 3.0f * 5.9604645e-08f;
    const float mr0 = 2.0f * rcr2f * 2.3841858e-07f, ma0 = 2.0f * rca2f * 2.3841858e-07f;
    const unsigned lt = (1u << lane) - 1u;
    int base = 0;
    for (int c0 = 0; c0 < nc; c0 += 32 * RF_UNROLL) {
        float4 pj[RF_UNROLL];
        if (c0 > 0) {
#pragma unroll
            for (int u = 0; u < RF_UNROLL; ++u) e[u] = (c0 + 32 * u + lane < nc) ? row[c0 + 32 * u + lane] : 0u;
        }
#pragma unroll
        for (int u = 0; u < RF_UNROLL; ++u) pj[u] = spos[(c0 + 32 * u + lane < nc) ? (e[u] & 0x0fffffffu) : i];
#pragma unroll
        for (int u = 0; u < RF_UNROLL; ++u) {
            if (c0 + 32 * u >= nc) break;                                  // warp-uniform
            const bool have = c0 + 32 * u + lane < nc;
            float dx = pj[u].x - pi.x, dy = pj[u].y - pi.y, dz = pj[u].z - pi.z;
            const float dm = fmaxf(fabsf(dx), fmaxf(fabsf(dy), fabsf(dz)));
            if (per) { dx -= Lx * rintf(dx * iLx); dy -= Ly * rintf(dy * iLy); dz -= Lz * rintf(dz * iLz); }
            const float r2 = dx * dx + dy * dy + dz * dz;
            bool in_r = have && r2 <= rcr2f;
            bool in_a = have && r2 <= rca2f;
            if (have && (fabsf(r2 - rcr2f) <= fmaf(kr, dm, mr0) || fabsf(r2 - rca2f) <= fmaf(ka, dm, ma0))) {
                const double r2d = pair_r2_box(pi, pj[u], bx);
                in_r = r2d <= rcr2;
                in_a = r2d <= rca2;
            }
            const unsigned m = __ballot_sync(0xffffffffu, in_r);
            if (in_r) {
                const int pos = base + __popc(m & lt);
                if (pos < stride) tmp[(size_t)i * stride + pos] = e[u] | (in_a ? 0u : ENT_RADIAL_ONLY);
            }
            base += __popc(m);
        }
    }
    if (lane == 0) {
        if (base > stride) { atomicExch(status, DHP_E_CAPACITY); base = stride; }
        cnt[i] = base;
        atomicAdd(&blk_sum[i / ROWS_PER_BLK], base);
    }
}

// ---------------------------------------------------------------------------------------------
// Small systems (n <= SMALL_N; the hybrid scheme's solute, BASELINE.json configs[0]-[1]).  The thirteen launches of the
// general path cost 3-15 us each, far more than their work; here a1 is three launches whose work is one warp per atom
// (round 1 did all of it in ONE block: 9 atoms per warp in sequence, each with several dependent global round trips -
// 61 us for 288 atoms; spread over n warps it is a few microseconds, and the launches cost nothing inside the replayed
// graph of the small-system call).  The atoms stay in the caller's order (perm = identity); every pair is tested (fp32
// with the error margin of k_refilter, the canonical fp64 predicate inside it: the list is the same bit-exact list):
//   k_small_pairs   warp <-> atom: all pairs of the row -> unordered entries (pass-1 format), counts; sorted copies
//   k_small_rows    warp <-> atom: CSR offset (prefix over at most 320 counts), order_row(): runs, masks
//   k_small_assign  one block: species-grouped, class-ordered row assignment (stable count over <= 320 keys), tile masks
// ---------------------------------------------------------------------------------------------
constexpr int SMALL_WARPS = 8;

__global__ void __launch_bounds__(SMALL_WARPS * 32)
k_small_pairs(const float* __restrict__ pos, const int* __restrict__ species, int n, const int* __restrict__ mol_offsets, int n_mol,
              const uint8_t* __restrict__ central, int periodic, double Lx, double Ly, double Lz, double rcr2, double rca2, int stride,
              Grid* __restrict__ grid, int* __restrict__ status, int* __restrict__ perm, int* __restrict__ inv_perm,
              float4* __restrict__ spos, int* __restrict__ smol, unsigned char* __restrict__ snc, unsigned* __restrict__ tmp,
              int* __restrict__ n_rad) {
    __shared__ Grid g;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const bool by_mol = mol_offsets != nullptr && n_mol > 0;
    if (tid == 0) {                                          // grid description (what the AEV kernels read)
        const double L[3] = {Lx, Ly, Lz};
        g.periodic = periodic; g.by_molecule = by_mol ? 1 : 0; g.ncell = 1;
        for (int c = 0; c < 3; ++c) {
            g.L[c] = periodic ? L[c] : 0.0; g.origin[c] = 0.0; g.inv_cell[c] = 0.0; g.nc[c] = 1; g.edge[c] = 0.0;
            g.inv_L[c] = periodic ? 1.0 / L[c] : 0.0; g.wrap[c] = periodic ? 1 : 0;
            g.Lf[c] = (float)L[c]; g.inv_Lf[c] = periodic ? (float)(1.0 / L[c]) : 0.f;
        }
        if (blockIdx.x == 0) *grid = g;
    }
    __syncthreads();
    const int i = blockIdx.x * SMALL_WARPS + warp;
    if (i >= n) return;
    auto mol_of = [&](int a) -> int {                        // largest m with mol_offsets[m] <= a
        if (!by_mol) return 0;
        int lo = 0, hi = n_mol;
        while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (mol_offsets[mid] <= a) lo = mid; else hi = mid; }
        return lo;
    };
    int si = species[i];
    if (lane == 0 && (si < 0 || si >= NSP)) atomicCAS(status, 0, DHP_E_SPECIES);
    si = min(max(si, 0), NSP - 1);
    const float4 pi = make_float4(pos[3 * i], pos[3 * i + 1], pos[3 * i + 2], __int_as_float(si));
    const int mi = mol_of(i);
    const unsigned char nci = central ? (central[i] ? 0 : 1) : 0;
    if (lane == 0) { spos[i] = pi; smol[i] = mi; snc[i] = nci; perm[i] = i; inv_perm[i] = i; }
    int base = 0;
    if (!nci) {
        const float rcr2f = (float)rcr2, rca2f = (float)rca2;
        const float rcr = sqrtf(rcr2f), rca = sqrtf(rca2f);
        const float kr = 2.0f * 2.0f * rcr * 3.0f * 5.9604645e-08f, ka = 2.0f * 2.0f * rca * 3.0f * 5.9604645e-08f;
        const float mr0 = 2.0f * rcr2f * 2.3841858e-07f, ma0 = 2.0f * rca2f * 2.3841858e-07f;
        const float Lfx = g.Lf[0], Lfy = g.Lf[1], Lfz = g.Lf[2], iLx = g.inv_Lf[0], iLy = g.inv_Lf[1], iLz = g.inv_Lf[2];
        const unsigned lt = (1u << lane) - 1u;
        for (int c0 = 0; c0 < n; c0 += 32) {
            const int j = c0 + lane, jc = min(j, n - 1);
            const int sj = min(max(species[jc], 0), NSP - 1);
            const float4 pj = make_float4(pos[3 * jc], pos[3 * jc + 1], pos[3 * jc + 2], __int_as_float(sj));
            const bool have = j < n && j != i && (!by_mol || mol_of(jc) == mi);
            float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
            const float dm = fmaxf(fabsf(dx), fmaxf(fabsf(dy), fabsf(dz)));
            if (periodic) { dx -= Lfx * rintf(dx * iLx); dy -= Lfy * rintf(dy * iLy); dz -= Lfz * rintf(dz * iLz); }
            const float r2 = dx * dx + dy * dy + dz * dz;
            bool in_r = have && r2 <= rcr2f;
            bool in_a = have && r2 <= rca2f;
            if (have && (fabsf(r2 - rcr2f) <= fmaf(kr, dm, mr0) || fabsf(r2 - rca2f) <= fmaf(ka, dm, ma0))) {
                const double r2d = pair_r2(pi, pj, g);
                in_r = r2d <= rcr2;
                in_a = r2d <= rca2;
            }
            const unsigned m = __ballot_sync(0xffffffffu, in_r);
            if (in_r) {
                const int o = base + __popc(m & lt);
                if (o < stride) tmp[(size_t)i * stride + o] = (unsigned)j | ((unsigned)sj << 28) | (in_a ? 0u : ENT_RADIAL_ONLY);
            }
            base += __popc(m);
        }
    }
    if (lane == 0) {
        if (base > stride) { atomicExch(status, DHP_E_CAPACITY); base = stride; }
        n_rad[i] = base;
    }
}

__global__ void __launch_bounds__(SMALL_WARPS * 32)
k_small_rows(const unsigned* __restrict__ tmp, int stride, const int* __restrict__ n_rad_in, int n, int64_t pair_cap,
             int* __restrict__ status, int* __restrict__ row_ptr, int* __restrict__ col, int* __restrict__ n_ang,
             unsigned short* __restrict__ seg_cnt, unsigned* __restrict__ amask) {
    __shared__ int segs[SMALL_WARPS][16];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int i = blockIdx.x * SMALL_WARPS + warp;
    if (i >= n) return;
    // CSR offset of row i and the total, from the (at most SMALL_N) counts: no separate scan launch
    int before = 0, total = 0;
    for (int a = lane; a < n; a += 32) { const int c = n_rad_in[a]; total += c; if (a < i) before += c; }
    for (int o = 16; o; o >>= 1) { before += __shfl_xor_sync(0xffffffffu, before, o); total += __shfl_xor_sync(0xffffffffu, total, o); }
    int ni = n_rad_in[i];
    if ((int64_t)total > pair_cap) {                         // neighbour storage overflow: an empty list, as in the general path
        if (lane == 0 && i == 0) atomicExch(status, DHP_E_CAPACITY);
        before = 0; total = 0; ni = 0;
    }
    __syncwarp();
    if (lane == 0) { row_ptr[i] = before; if (i == n - 1) row_ptr[n] = total; }
    order_row(tmp + (size_t)i * stride, ni, before, i, lane, lane_pair_species(lane), segs[warp], col, n_ang, seg_cnt, amask, false, nullptr, nullptr);
}

constexpr int SMALL_THREADS = 320;
static_assert(SMALL_THREADS >= SMALL_N, "one thread per atom in k_small_assign");

__global__ void __launch_bounds__(SMALL_THREADS)
k_small_assign(const float4* __restrict__ spos, const unsigned char* __restrict__ snc, const unsigned* __restrict__ amask, int n,
               const int* __restrict__ row_ptr, int* __restrict__ n_rad, int* __restrict__ sp_count, int* __restrict__ sp_start, int* __restrict__ rowmap, int* __restrict__ row_species,
               int* __restrict__ row_slot, unsigned* __restrict__ tile_mask) {
    __shared__ short key_s[SMALL_N];
    __shared__ int tot_s[NKEY], kstart_s[NKEY];
    const int tid = threadIdx.x;
    for (int k = tid; k < NKEY; k += SMALL_THREADS) tot_s[k] = 0;
    if (tid < n && row_ptr[n] == 0) n_rad[tid] = 0;          // an emptied (overflowed) list: the counts the export reads say so too
    int key = -1, sp = 0;
    unsigned am = 0;
    if (tid < n && !snc[tid]) { sp = __float_as_int(spos[tid].w); am = amask[tid]; key = row_key(sp, am); }
    if (tid < n) key_s[tid] = (short)key;
    __syncthreads();
    int rank = 0;
    if (key >= 0) {
        int same = 0;
        for (int b = 0; b < n; ++b) {
            const bool eq = key_s[b] == (short)key;
            same += eq;
            rank += eq && b < tid;
        }
        if (rank == 0) tot_s[key] = same;
    }
    __syncthreads();
    if (tid == 0) {
        int start = 0;
        for (int s = 0; s < NSP; ++s) {
            sp_start[s] = start;
            int c = 0;
            for (int k = 0; k < NCLS; ++k) { kstart_s[s * NCLS + k] = start + c; c += tot_s[s * NCLS + k]; }
            sp_count[s] = c;
            start += (c + ROW_ALIGN - 1) / ROW_ALIGN * ROW_ALIGN;
        }
        sp_start[NSP] = start;
        sp_count[NSP] = 0;
    }
    __syncthreads();
    if (tid < n) {
        if (key < 0) { rowmap[tid] = -1; return; }
        const int row = kstart_s[key] + rank;
        rowmap[tid] = row;
        row_species[row] = sp;
        row_slot[row] = tid;
        if (am) { atomicOr(&tile_mask[(row / ROW_TILE) & ~1], am); atomicOr(&tile_mask[(row / ROW_TILE) | 1], am); }
    }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
// List reuse (dhp_set_skin): is this call the same problem as the one the candidate list was built for (size, box, molecule
// table, masked or not)?  Whether the atoms have stayed within skin / 2 is decided on the device.  Shared with the graph replay
// of the hot call (api.cu), which must pick the graph of the right enqueue (reuse check, or forced rebuild) and leave the same
// host-side record behind as a plain enqueue.
static void reuse_box(const float* box_host, float (&bx)[4]) {
    const bool periodic = box_host != nullptr;
    for (int c = 0; c < 3; ++c) bx[c] = periodic ? (float)(double)box_host[c] : 0.f;
    bx[3] = periodic ? 1.f : 0.f;
}
bool nlist_reuse_same(const Ctx* ctx, int64_t n, const float* box_host, const int32_t* mol_offsets, int64_t n_mol, const uint8_t* central) {
    const bool by_mol = mol_offsets != nullptr && n_mol > 0;
    float bx[4];
    reuse_box(box_host, bx);
    return ctx->cand_valid && ctx->cand_n == n && ctx->cand_nmol == (by_mol ? n_mol : 0) && ctx->cand_mol == (const void*)mol_offsets &&
           ctx->cand_central == (central != nullptr) && memcmp(bx, ctx->cand_box, sizeof(bx)) == 0;
}
void nlist_reuse_mark(Ctx* ctx, int64_t n, const float* box_host, const int32_t* mol_offsets, int64_t n_mol, const uint8_t* central) {
    const bool by_mol = mol_offsets != nullptr && n_mol > 0;
    float bx[4];
    reuse_box(box_host, bx);
    ctx->cand_valid = true; ctx->cand_n = n; ctx->cand_nmol = by_mol ? n_mol : 0; ctx->cand_mol = (const void*)mol_offsets;
    ctx->cand_central = central != nullptr; memcpy(ctx->cand_box, bx, sizeof(bx));
}

int nlist_build(Ctx* ctx, const float* pos, const float* box_host, const int32_t* species, int64_t n64,
                const int32_t* mol_offsets, int64_t n_mol64, const uint8_t* central) {
    const int n = (int)n64, n_mol = (int)n_mol64;
    const bool periodic = box_host != nullptr;
    const bool by_mol = mol_offsets != nullptr && n_mol > 0;
    const double rcr = (double)ctx->params.rcr, rca = (double)ctx->params.rca;
    ctx->n_atoms = n;
    ctx->n_mol = by_mol ? n_mol : 0;
    ctx->periodic = periodic;
    ctx->partial = central != nullptr;
    const unsigned char* snc = central ? ctx->snc : nullptr;
    cudaStream_t st = ctx->stream;
    const int nblk = (n + ROWS_PER_BLK - 1) / ROWS_PER_BLK;
    const bool skin = ctx->skin > 0.f && ctx->cand != nullptr && n > 0;
    const int* gate = skin ? ctx->rebuild : nullptr;             // nullptr: every kernel of the build path runs
    const double rl = rcr + (skin ? (double)ctx->skin : 0.0);    // list radius: the cell grid must cover it

    // one memset zeroes everything this call accumulates into (status word, cell counters, tile masks, block sums, and for
    // the later phases the tile schedulers, atomic energies and sorted forces), one sets the row tables to -1
    DHP_CUDA(ctx, cudaMemsetAsync(ctx->zero_arena, 0, sizeof(unsigned) * ctx->zero_words, st));
    if (!skin) {
        DHP_CUDA(ctx, cudaMemsetAsync(ctx->ff_arena, 0xFF, sizeof(int) * 2 * ctx->max_rows, st));
        ctx->cand_valid = false;
    }
    if (n == 0) {
        DHP_CUDA(ctx, cudaMemsetAsync(ctx->row_ptr, 0, sizeof(int), st));
        DHP_CUDA(ctx, cudaMemsetAsync(ctx->sp_count, 0, sizeof(int) * 8, st));
        DHP_CUDA(ctx, cudaMemsetAsync(ctx->sp_start, 0, sizeof(int) * 8, st));
        ctx->cand_valid = false;
        return DHP_OK;
    }
    double L[3] = {0, 0, 0};
    if (periodic) for (int c = 0; c < 3; ++c) L[c] = (double)box_host[c];
    if (!skin && n <= SMALL_N && !ctx->no_small_path) {          // small systems: the whole of a1 in one block
        const int sb = (n + SMALL_WARPS - 1) / SMALL_WARPS;
        DHP_LAUNCH(ctx, k_small_pairs, sb, SMALL_WARPS * 32, 0, pos, species, n, mol_offsets, by_mol ? n_mol : 0, central, periodic ? 1 : 0,
                   L[0], L[1], L[2], rcr * rcr, rca * rca, ctx->tmp_stride, ctx->grid, ctx->status, ctx->perm, ctx->inv_perm, ctx->spos,
                   ctx->smol, ctx->snc, ctx->tmp_col, ctx->n_rad);
        DHP_LAUNCH(ctx, k_small_rows, sb, SMALL_WARPS * 32, 0, ctx->tmp_col, ctx->tmp_stride, ctx->n_rad, n, ctx->pair_cap, ctx->status,
                   ctx->row_ptr, ctx->col, ctx->n_ang, ctx->seg_cnt, ctx->amask);
        DHP_LAUNCH(ctx, k_small_assign, 1, SMALL_THREADS, 0, ctx->spos, ctx->snc, ctx->amask, n, ctx->row_ptr, ctx->n_rad, ctx->sp_count, ctx->sp_start, ctx->rowmap,
                   ctx->row_species, ctx->row_slot, ctx->tile_mask);
        DHP_CUDA(ctx, cudaGetLastError());
        return DHP_OK;
    }
    const int nb = (n + 255) / 256;
    if (skin) {
        // reuse is possible only for the same problem (size, box, molecule table, masked or not); whether the atoms
        // have stayed within skin / 2 of the last full build is decided on the device
        const float bx[4] = {(float)L[0], (float)L[1], (float)L[2], periodic ? 1.f : 0.f};
        const bool same = nlist_reuse_same(ctx, n, box_host, mol_offsets, n_mol, central);
        if (same) {
            DHP_CUDA(ctx, cudaMemsetAsync(ctx->rebuild, 0, sizeof(int), st));
            const float h = 0.5f * ctx->skin;
            DHP_LAUNCH(ctx, k_reuse_check, nb, 256, 0, pos, species, ctx->pos_ref, ctx->spos, ctx->inv_perm, central, ctx->snc, n,
                       h * h * 0.9999f, ctx->rebuild, ctx->cand_bad, by_mol ? mol_offsets : (const int32_t*)nullptr, ctx->smol);
        } else {
            DHP_LAUNCH(ctx, k_set_flag, 1, 1, 0, ctx->rebuild, 1);
        }
        (void)bx;
        nlist_reuse_mark(ctx, n, box_host, mol_offsets, n_mol, central);
        DHP_LAUNCH(ctx, k_reset_rows, 2 * ctx->sm_count, 256, 0, ctx->row_slot, ctx->row_species, (int)ctx->max_rows, gate);
    }
    if (!periodic && !by_mol) {
        // ordered-uint min / max accumulators: {0xffffffff x 3, 0 x 3} (two memsets: a copy from pageable host memory could
        // not be captured into a CUDA graph)
        DHP_CUDA(ctx, cudaMemsetAsync(ctx->bbox, 0xFF, 3 * sizeof(unsigned), st));
        DHP_CUDA(ctx, cudaMemsetAsync(ctx->bbox + 3, 0, 3 * sizeof(unsigned), st));
        int blocks = (int)std::min<int64_t>((n + 255) / 256, 4 * ctx->sm_count);
        DHP_LAUNCH(ctx, k_bbox, blocks, 256, 0, pos, n, ctx->bbox, gate);
    }
    DHP_LAUNCH(ctx, k_setup_grid, 1, 32, 0, ctx->grid, periodic ? 1 : 0, L[0], L[1], L[2], rl, ctx->bbox,
               (int)ctx->max_cells, by_mol ? 1 : 0, n_mol, gate, skin ? ctx->rebuild_count : (int*)nullptr, ctx->cand_bad);
    DHP_LAUNCH(ctx, k_assign_cells, nb, 256, 0, pos, species, n, mol_offsets, n_mol, ctx->grid, ctx->cell_of,
               ctx->cell_count, ctx->status, gate);
    DHP_LAUNCH(ctx, k_scan_cells, 1, 1024, 0, ctx->cell_count, ctx->cell_start, ctx->grid, gate);
    DHP_LAUNCH(ctx, k_scatter, nb, 256, 0, ctx->cell_of, n, ctx->cell_start, ctx->cell_fill, ctx->perm_tmp, gate);
    // the cell count lives on the device; launch for the bound and let surplus blocks exit
    int64_t cell_bound = by_mol ? n_mol : ctx->max_cells;
    if (periodic) {
        int64_t t = 1;
        for (int c = 0; c < 3; ++c) t *= (int64_t)fmax(1.0, floor(L[c] / rl));
        cell_bound = t < cell_bound ? t : cell_bound;
    }
    DHP_LAUNCH(ctx, k_sort_gather, (int)((cell_bound + 3) / 4), 128, 0, pos, species, ctx->grid, ctx->cell_start,
               ctx->perm_tmp, ctx->perm, ctx->inv_perm, ctx->spos, ctx->smol, central, ctx->snc, gate,
               skin ? ctx->pos_ref : (float*)nullptr);
    // pair list
    const double rcr2 = rcr * rcr, rca2 = rca * rca;
    bool wrap = false;     // same rule as k_setup_grid: a periodic axis with fewer than 3 cells
    if (periodic) {
        const double edge = rl * (1.0 + 9.5367431640625e-07);
        for (int c = 0; c < 3; ++c) wrap |= floor(L[c] / edge) < 3.0;
        // k_setup_grid may coarsen the grid when it exceeds max_cells; be conservative then
        if ((double)floor(L[0] / edge) * floor(L[1] / edge) * floor(L[2] / edge) > (double)ctx->max_cells) wrap = true;
    }
    const float rs2f = (float)(rl * rl);
#define DHP_PAIRS(W, S)                                                                                                        \
    DHP_LAUNCH(ctx, (k_pairs<W, S>), (int)cell_bound, P1_THREADS, 0, ctx->spos, ctx->grid, ctx->cell_start, rcr2, rca2,       \
               ctx->tmp_stride, ctx->n_rad, ctx->tmp_col, ctx->blk_sum, ctx->status, snc, gate, rs2f, ctx->cand_stride,       \
               ctx->cand_cnt, ctx->cand)
    if (wrap) { if (skin) DHP_PAIRS(true, true); else DHP_PAIRS(true, false); }
    else      { if (skin) DHP_PAIRS(false, true); else DHP_PAIRS(false, false); }
#undef DHP_PAIRS
    if (skin) {
        DHP_LAUNCH(ctx, k_regather, nb, 256, 0, pos, ctx->perm, n, ctx->spos, gate);
        BoxArg bxa;
        for (int c = 0; c < 3; ++c) { bxa.L[c] = L[c]; bxa.Lf[c] = (float)L[c]; bxa.iLf[c] = periodic ? (float)(1.0 / L[c]) : 0.f; }
        bxa.periodic = periodic ? 1 : 0;
        DHP_LAUNCH(ctx, k_refilter, (n + RF_WARPS - 1) / RF_WARPS, RF_WARPS * 32, 0, ctx->spos, bxa, ctx->cand, ctx->cand_cnt,
                   ctx->cand_stride, rcr2, rca2, ctx->tmp_stride, n, ctx->n_rad, ctx->tmp_col, ctx->blk_sum, ctx->status, snc, gate);
    }
    DHP_LAUNCH(ctx, k_scan_blocks, 1, 1024, 0, ctx->blk_sum, ctx->blk_off, nblk, ctx->pair_cap, ctx->status, ctx->cand_bad);
    DHP_LAUNCH(ctx, k_rows, nblk, P2_THREADS, 0, ctx->tmp_col, ctx->tmp_stride, ctx->n_rad, ctx->blk_off, nblk, n, ctx->row_ptr,
               ctx->col, ctx->n_rad, ctx->n_ang, ctx->seg_cnt, ctx->amask, gate, ctx->rowmap, ctx->tile_mask);
    // rows grouped by species, ordered by feature-block class inside a group; tile masks
    const int nrb = (n + RB - 1) / RB;
    DHP_LAUNCH(ctx, k_rowkey_hist, nrb, RB, 0, ctx->spos, ctx->amask, snc, n, nrb, ctx->blk_hist, gate);
    DHP_LAUNCH(ctx, k_rowkey_scan, NSP, 1024, 0, ctx->blk_hist, nrb, ctx->sp_count, ctx->sp_start, ctx->key_start, ctx->rowkey_done, gate);
    DHP_LAUNCH(ctx, k_rowkey_rank, nrb, RB, 0, ctx->spos, ctx->amask, snc, n, nrb, ctx->blk_hist, ctx->key_start, ctx->rowmap,
               ctx->row_species, ctx->row_slot, ctx->tile_mask, gate);
    DHP_CUDA(ctx, cudaGetLastError());
    return DHP_OK;
}

// ---------------------------------------------------------------------------------------------
// canonical export (test / interface use; not on the hot path)
// ---------------------------------------------------------------------------------------------
__global__ void k_export_counts(const int* __restrict__ inv_perm, const int* __restrict__ n_rad,
                                const int* __restrict__ n_ang, int n, int angular, int* __restrict__ out) {
    int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a < n) out[a] = angular ? n_ang[inv_perm[a]] : n_rad[inv_perm[a]];
}
__global__ void k_scan_n(const int* __restrict__ in, int* __restrict__ out, int n) { block_scan_excl(in, out, n); }

__global__ void k_export_fill(const int* __restrict__ inv_perm, const int* __restrict__ perm,
                              const int* __restrict__ row_ptr, const int* __restrict__ col, int n,
                              const int* __restrict__ rp_out, int* __restrict__ col_out) {
    int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= n) return;
    int src = row_ptr[inv_perm[a]];
    int b = rp_out[a], e = rp_out[a + 1];
    for (int t = b; t < e; ++t) {          // insertion sort into ascending caller indices
        int v = perm[col[src + (t - b)]];
        int q = t - 1;
        while (q >= b && col_out[q] > v) { col_out[q + 1] = col_out[q]; --q; }
        col_out[q + 1] = v;
    }
}

int nlist_export(Ctx* ctx, int32_t* row_ptr_out, int32_t* col_out, bool angular) {
    const int n = (int)ctx->n_atoms;
    if (n == 0) {
        DHP_CUDA(ctx, cudaMemsetAsync(row_ptr_out, 0, sizeof(int), ctx->stream));
        return DHP_OK;
    }
    const int nb = (n + 127) / 128;
    DHP_LAUNCH(ctx, k_export_counts, nb, 128, 0, ctx->inv_perm, ctx->n_rad, ctx->n_ang, n, angular ? 1 : 0,
               ctx->export_tmp);
    DHP_LAUNCH(ctx, k_scan_n, 1, 1024, 0, ctx->export_tmp, row_ptr_out, n);
    if (col_out)
        DHP_LAUNCH(ctx, k_export_fill, nb, 128, 0, ctx->inv_perm, ctx->perm, ctx->row_ptr, ctx->col, n, row_ptr_out,
                   col_out);
    DHP_CUDA(ctx, cudaGetLastError());
    return DHP_OK;
}

}  // namespace dhp
