// a1 — neighbour search: periodic / open cell list -> CSR pair list (§2.2.2).
//
// Atoms are binned into cells of edge >= rc(1+2^-20), counting-sorted by cell (ties broken by the
// caller's index, so the internal order is deterministic), and each atom's stencil of <= 27 cells is
// scanned twice (count, then fill).  The keep/drop decision is ONLY the canonical fp64 predicate of
// include/dhp.h: binning is conservative, never decisive.  Rows hold sorted-slot
// indices with the angular neighbours (R <= rca) as a prefix.  Rows of the AEV / MLP buffers are
// grouped by the central atom's species (stable in sorted order), each group starting at a multiple
// of ROW_TILE rows so that one MLP tile never mixes networks.
#include <algorithm>

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

// exclusive scan of n ints by ONE block of 1024 threads; out[n] = total
__device__ void block_scan_excl(const int* __restrict__ in, int* __restrict__ out, int n) {
    __shared__ int warp_sums[32];
    __shared__ int carry_s;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) carry_s = 0;
    __syncthreads();
    for (int base = 0; base < n; base += 1024) {
        int idx = base + tid;
        int v = idx < n ? in[idx] : 0;
        int x = v;
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
        int carry = carry_s;
        int excl = carry + (wid ? warp_sums[wid - 1] : 0) + x - v;
        if (idx < n) out[idx] = excl;
        __syncthreads();
        if (tid == 1023) carry_s = carry + warp_sums[31];
        __syncthreads();
    }
    if (tid == 0) out[n] = carry_s;
}

// ---------------------------------------------------------------------------------------------
// grid setup
// ---------------------------------------------------------------------------------------------
__global__ void k_bbox(const float* __restrict__ pos, int n, unsigned* __restrict__ bbox) {
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
                             const unsigned* __restrict__ bbox, int max_cells, int by_molecule, int n_mol) {
    if (threadIdx.x || blockIdx.x) return;
    const double edge = rc * (1.0 + 9.5367431640625e-07);   // rc (1 + 2^-20): binning slack
    double L[3] = {Lx, Ly, Lz};
    g->periodic = periodic;
    g->by_molecule = by_molecule;
    if (by_molecule) {
        for (int c = 0; c < 3; ++c) { g->L[c] = 0; g->origin[c] = 0; g->inv_cell[c] = 0; g->nc[c] = 1; }
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
    for (int c = 0; c < 3; ++c) g->inv_cell[c] = (double)g->nc[c] / ext[c];
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
                               int* __restrict__ cell_of, int* __restrict__ cell_count, int* __restrict__ status) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int s = species[i];
    if (s < 0 || s >= NSP) atomicExch(status, DHP_E_SPECIES);
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

__global__ void k_scan_cells(const int* __restrict__ cnt, int* __restrict__ start, const Grid* __restrict__ g) {
    block_scan_excl(cnt, start, g->ncell);
}

__global__ void k_scatter(const int* __restrict__ cell_of, int n, const int* __restrict__ cell_start,
                          int* __restrict__ cell_fill, int* __restrict__ perm) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int c = cell_of[i];
    perm[cell_start[c] + atomicAdd(&cell_fill[c], 1)] = i;
}

// one thread per cell: order its atoms by caller index (deterministic internal order), then gather
__global__ void k_sort_gather(const float* __restrict__ pos, const int* __restrict__ species,
                              const Grid* __restrict__ g, const int* __restrict__ cell_start, int* __restrict__ perm,
                              int* __restrict__ inv_perm, float4* __restrict__ spos, int* __restrict__ smol,
                              int* __restrict__ scell) {
    int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= g->ncell) return;
    int b = cell_start[c], e = cell_start[c + 1];
    for (int a = b + 1; a < e; ++a) {
        int v = perm[a], q = a - 1;
        while (q >= b && perm[q] > v) { perm[q + 1] = perm[q]; --q; }
        perm[q + 1] = v;
    }
    for (int a = b; a < e; ++a) {
        int i = perm[a];
        inv_perm[i] = a;
        int s = species[i];
        s = min(max(s, 0), NSP - 1);
        spos[a] = make_float4(pos[3 * i], pos[3 * i + 1], pos[3 * i + 2], __int_as_float(s));
        smol[a] = g->by_molecule ? c : 0;
        scell[a] = c;
    }
}

// ---------------------------------------------------------------------------------------------
// species-grouped rows (stable in sorted order)
// ---------------------------------------------------------------------------------------------
constexpr int RB = 256;   // slots per block in the row assignment

__global__ void k_species_hist(const float4* __restrict__ spos, int n, int* __restrict__ blk_hist) {
    __shared__ int h[NSP];
    if (threadIdx.x < NSP) h[threadIdx.x] = 0;
    __syncthreads();
    int a = blockIdx.x * RB + threadIdx.x;
    int s = a < n ? __float_as_int(spos[a].w) : -1;
    for (int t = 0; t < NSP; ++t) {
        unsigned m = __ballot_sync(0xffffffffu, s == t);
        if ((threadIdx.x & 31) == 0 && m) atomicAdd(&h[t], __popc(m));
    }
    __syncthreads();
    if (threadIdx.x < NSP) blk_hist[blockIdx.x * 8 + threadIdx.x] = h[threadIdx.x];
}

// single block: per species exclusive scan over blocks; group starts aligned to ROW_TILE
__global__ void k_species_scan(int* __restrict__ blk_hist, int nblk, int* __restrict__ sp_count, int* __restrict__ sp_start) {
    __shared__ int tot[NSP + 1];
    int t = threadIdx.x;
    if (t < NSP) {
        int run = 0;
        for (int b = 0; b < nblk; ++b) {
            int v = blk_hist[b * 8 + t];
            blk_hist[b * 8 + t] = run;
            run += v;
        }
        tot[t] = run;
    }
    __syncthreads();
    if (t == 0) {
        int start = 0;
        for (int s = 0; s < NSP; ++s) {
            sp_count[s] = tot[s];
            sp_start[s] = start;
            start += (tot[s] + ROW_TILE - 1) / ROW_TILE * ROW_TILE;
        }
        sp_start[NSP] = start;
        sp_count[NSP] = 0;
    }
}

__global__ void k_species_rank(const float4* __restrict__ spos, int n, const int* __restrict__ blk_hist,
                               const int* __restrict__ sp_start, int* __restrict__ rowmap,
                               int* __restrict__ row_species, int* __restrict__ row_slot) {
    __shared__ int wcnt[RB / 32][NSP];
    int a = blockIdx.x * RB + threadIdx.x;
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int s = a < n ? __float_as_int(spos[a].w) : -1;
    int rank_in_warp = 0;
    for (int t = 0; t < NSP; ++t) {
        unsigned m = __ballot_sync(0xffffffffu, s == t);
        if (s == t) rank_in_warp = __popc(m & ((1u << lane) - 1u));
        if (lane == 0) wcnt[w][t] = __popc(m);
    }
    __syncthreads();
    if (a >= n) return;
    int before = 0;
    for (int q = 0; q < w; ++q) before += wcnt[q][s];
    int row = sp_start[s] + blk_hist[blockIdx.x * 8 + s] + before + rank_in_warp;
    rowmap[a] = row;
    row_species[row] = s;
    row_slot[row] = a;
}

// ---------------------------------------------------------------------------------------------
// stencil traversal (count + fill share it)
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

template <bool FILL>
__global__ void __launch_bounds__(256) k_neighbours(const float4* __restrict__ spos, const int* __restrict__ scell, int n,
                                                   const Grid* __restrict__ gp, const int* __restrict__ cell_start,
                                                   double rcr2, double rca2, int* __restrict__ n_rad,
                                                   int* __restrict__ n_ang, const int* __restrict__ row_ptr,
                                                   int* __restrict__ col) {
    __shared__ Grid g;
    if (threadIdx.x == 0) g = *gp;
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (i >= n) return;
    const float4 pi = spos[i];
    Stencil st;
    make_stencil(g, scell[i], st);
    int cnt_r = 0, cnt_a = 0;
    int base_a = 0, base_r = 0;
    if (FILL) {
        base_a = row_ptr[i];
        base_r = base_a + n_ang[i];
        if (row_ptr[i + 1] - base_a != n_rad[i]) return;   // overflowed list was emptied by the scan
    }
    const unsigned lt = (1u << lane) - 1u;
    for (int iz = 0; iz < st.n[2]; ++iz)
        for (int iy = 0; iy < st.n[1]; ++iy)
            for (int ix = 0; ix < st.n[0]; ++ix) {
                int c = g.by_molecule ? st.c[0][0] : st.c[0][ix] + g.nc[0] * (st.c[1][iy] + g.nc[1] * st.c[2][iz]);
                int b = cell_start[c], e = cell_start[c + 1];
                for (int j0 = b; j0 < e; j0 += 32) {
                    int j = j0 + lane;
                    bool in_r = false, in_a = false;
                    if (j < e && j != i) {
                        double r2 = pair_r2(pi, spos[j], g);
                        in_r = r2 <= rcr2;
                        in_a = r2 <= rca2;
                    }
                    if (FILL) {
                        unsigned ma = __ballot_sync(0xffffffffu, in_a);
                        unsigned mr = __ballot_sync(0xffffffffu, in_r && !in_a);
                        if (in_a) col[base_a + __popc(ma & lt)] = j;
                        else if (in_r) col[base_r + __popc(mr & lt)] = j;
                        base_a += __popc(ma);
                        base_r += __popc(mr);
                    } else {
                        cnt_r += in_r;
                        cnt_a += in_a;
                    }
                }
            }
    if (!FILL) {
        for (int o = 16; o; o >>= 1) {
            cnt_r += __shfl_xor_sync(0xffffffffu, cnt_r, o);
            cnt_a += __shfl_xor_sync(0xffffffffu, cnt_a, o);
        }
        if (lane == 0) { n_rad[i] = cnt_r; n_ang[i] = cnt_a; }
    }
}

__global__ void k_scan_rows(const int* __restrict__ n_rad, int* __restrict__ row_ptr, int n, int64_t pair_cap,
                            int* __restrict__ status) {
    __shared__ int overflow;
    block_scan_excl(n_rad, row_ptr, n);
    __syncthreads();
    if (threadIdx.x == 0) {
        // int32 wrap-around shows up as a negative or non-monotone total; both count as overflow
        overflow = (row_ptr[n] < 0 || (int64_t)row_ptr[n] > pair_cap) ? 1 : 0;
        if (overflow) atomicExch(status, DHP_E_CAPACITY);
    }
    __syncthreads();
    if (overflow)
        for (int i = threadIdx.x; i <= n; i += blockDim.x) row_ptr[i] = 0;
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
int nlist_build(Ctx* ctx, const float* pos, const float* box_host, const int32_t* species, int64_t n64,
                const int32_t* mol_offsets, int64_t n_mol64) {
    const int n = (int)n64, n_mol = (int)n_mol64;
    const bool periodic = box_host != nullptr;
    const bool by_mol = mol_offsets != nullptr && n_mol > 0;
    const double rcr = (double)ctx->params.rcr, rca = (double)ctx->params.rca;
    ctx->n_atoms = n;
    ctx->n_mol = by_mol ? n_mol : 0;
    ctx->periodic = periodic;
    cudaStream_t st = ctx->stream;

    DHP_CUDA(ctx, cudaMemsetAsync(ctx->status, 0, sizeof(int), st));
    DHP_CUDA(ctx, cudaMemsetAsync(ctx->cell_count, 0, sizeof(int) * (ctx->max_cells + 1), st));
    DHP_CUDA(ctx, cudaMemsetAsync(ctx->cell_fill, 0, sizeof(int) * ctx->max_cells, st));
    DHP_CUDA(ctx, cudaMemsetAsync(ctx->row_slot, 0xFF, sizeof(int) * ctx->max_rows, st));
    DHP_CUDA(ctx, cudaMemsetAsync(ctx->row_species, 0xFF, sizeof(int) * ctx->max_rows, st));
    if (n == 0) {
        DHP_CUDA(ctx, cudaMemsetAsync(ctx->row_ptr, 0, sizeof(int), st));
        DHP_CUDA(ctx, cudaMemsetAsync(ctx->sp_count, 0, sizeof(int) * 8, st));
        DHP_CUDA(ctx, cudaMemsetAsync(ctx->sp_start, 0, sizeof(int) * 8, st));
        return DHP_OK;
    }
    double L[3] = {0, 0, 0};
    if (periodic) for (int c = 0; c < 3; ++c) L[c] = (double)box_host[c];
    if (!periodic && !by_mol) {
        static const unsigned init[6] = {0xffffffffu, 0xffffffffu, 0xffffffffu, 0u, 0u, 0u};
        DHP_CUDA(ctx, cudaMemcpyAsync(ctx->bbox, init, sizeof(init), cudaMemcpyHostToDevice, st));
        int blocks = (int)std::min<int64_t>((n + 255) / 256, 4 * ctx->sm_count);
        DHP_LAUNCH(ctx, k_bbox, blocks, 256, 0, pos, n, ctx->bbox);
    }
    DHP_LAUNCH(ctx, k_setup_grid, 1, 32, 0, ctx->grid, periodic ? 1 : 0, L[0], L[1], L[2], rcr, ctx->bbox,
               (int)ctx->max_cells, by_mol ? 1 : 0, n_mol);
    const int nb = (n + 255) / 256;
    DHP_LAUNCH(ctx, k_assign_cells, nb, 256, 0, pos, species, n, mol_offsets, n_mol, ctx->grid, ctx->cell_of,
               ctx->cell_count, ctx->status);
    DHP_LAUNCH(ctx, k_scan_cells, 1, 1024, 0, ctx->cell_count, ctx->cell_start, ctx->grid);
    DHP_LAUNCH(ctx, k_scatter, nb, 256, 0, ctx->cell_of, n, ctx->cell_start, ctx->cell_fill, ctx->perm);
    // the cell count lives on the device; launch for the bound and let surplus threads exit
    int64_t cell_bound = by_mol ? n_mol : ctx->max_cells;
    if (periodic) {
        int64_t t = 1;
        for (int c = 0; c < 3; ++c) t *= (int64_t)fmax(1.0, floor(L[c] / rcr));
        cell_bound = t < cell_bound ? t : cell_bound;
    }
    DHP_LAUNCH(ctx, k_sort_gather, (int)((cell_bound + 127) / 128), 128, 0, pos, species, ctx->grid, ctx->cell_start,
               ctx->perm, ctx->inv_perm, ctx->spos, ctx->smol, ctx->scell);
    // rows grouped by species
    const int nrb = (n + RB - 1) / RB;
    DHP_LAUNCH(ctx, k_species_hist, nrb, RB, 0, ctx->spos, n, ctx->blk_hist);
    DHP_LAUNCH(ctx, k_species_scan, 1, 32, 0, ctx->blk_hist, nrb, ctx->sp_count, ctx->sp_start);
    DHP_LAUNCH(ctx, k_species_rank, nrb, RB, 0, ctx->spos, n, ctx->blk_hist, ctx->sp_start, ctx->rowmap,
               ctx->row_species, ctx->row_slot);
    // CSR
    const int nwb = (n + 7) / 8;   // 8 warps per block, one warp per atom
    const double rcr2 = rcr * rcr, rca2 = rca * rca;
    DHP_LAUNCH(ctx, k_neighbours<false>, nwb, 256, 0, ctx->spos, ctx->scell, n, ctx->grid, ctx->cell_start, rcr2,
               rca2, ctx->n_rad, ctx->n_ang, ctx->row_ptr, ctx->col);
    DHP_LAUNCH(ctx, k_scan_rows, 1, 1024, 0, ctx->n_rad, ctx->row_ptr, n, ctx->pair_cap, ctx->status);
    DHP_LAUNCH(ctx, k_neighbours<true>, nwb, 256, 0, ctx->spos, ctx->scell, n, ctx->grid, ctx->cell_start, rcr2,
               rca2, ctx->n_rad, ctx->n_ang, ctx->row_ptr, ctx->col);
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
