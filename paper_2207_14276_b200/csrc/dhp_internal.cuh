// Internal declarations shared by the translation units of libdhp.so (CUDA path only; the fp64
// oracle under oracle/ shares nothing with this directory).
#pragma once

#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/dhp.h"

namespace dhp {

constexpr int NSP = DHP_N_SPECIES;
constexpr int NR = DHP_N_SHF_R;
constexpr int NA = DHP_N_SHF_A;
constexpr int NZ = DHP_N_SHF_Z;
constexpr int NPAIR = NSP * (NSP + 1) / 2;      // 28
constexpr int AEV_RAD = NSP * NR;               // 112
constexpr int AEV_ANG = NPAIR * NA * NZ;        // 896
constexpr int AEV_DIM = AEV_RAD + AEV_ANG;      // 1008
constexpr int AEV_LD = 1024;                    // row pitch of AEV / dE/dAEV buffers (floats)
constexpr int H1 = 256, H2 = 192, H3 = 160;     // hidden widths (BASELINE.json configs[0])
constexpr int NET_PARAMS = DHP_NET_PARAMS;
constexpr int OFF_W1 = 0;
constexpr int OFF_B1 = OFF_W1 + AEV_DIM * H1;
constexpr int OFF_W2 = OFF_B1 + H1;
constexpr int OFF_B2 = OFF_W2 + H1 * H2;
constexpr int OFF_W3 = OFF_B2 + H2;
constexpr int OFF_B3 = OFF_W3 + H2 * H3;
constexpr int OFF_W4 = OFF_B3 + H3;
constexpr int OFF_B4 = OFF_W4 + H3;
static_assert(OFF_B4 + 1 == NET_PARAMS, "blob layout");

constexpr int ROW_TILE = 128;                   // rows of one MLP tile (UMMA M of one CTA)
constexpr int ROW_ALIGN = 2 * ROW_TILE;         // species groups start at multiples of this many rows: the two row tiles of a
                                                // CTA pair (tcgen05 cta_group::2) always run the same network; tile masks are
                                                // kept equal within such a pair
constexpr int KBLK = 64;                        // feature-block width: the unit in which zero columns are skipped
constexpr int N_KBLK = AEV_LD / KBLK;           // 16 blocks: 14 angular (2 species pairs each) + 2 radial
// The fp16 hi / lo planes of the AEV rows are stored in the tiled operand layout of the tensor path (mlp_tc.cu): the image
// of the no-swizzle K-major UMMA A tile, [plane][row tile][64-column block][8-column group][row in tile][8 halves], so that
// one 16-wide K step of a row tile is 4 KB of contiguous bytes per plane.  Offset in halves inside one plane:
__host__ __device__ __forceinline__ size_t aev_tiled_off(int row, int col) {
    return ((size_t)(row / ROW_TILE) * N_KBLK + (size_t)(col / KBLK)) * (size_t)(ROW_TILE * KBLK) +
           (size_t)((((col % KBLK) >> 3) * ROW_TILE + (row % ROW_TILE)) * 8 + (col & 7));
}
constexpr int SMALL_N = 320;                      // systems up to this size take the single-block list build (above ~300 atoms one SM is
                                                // slower than the thirteen small launches of the general path) and CUDA-graph replay
constexpr int MAX_MODELS = DHP_MAX_MODELS;
constexpr int MAX_ANG = DHP_MAX_ANG;                    // angular neighbours staged per centre (status CAPACITY beyond)

// Device-side description of the cell grid, written by a setup kernel (periodic: from host box;
// open: from the bounding box reduction) so that no hot call needs a host round trip.
struct Grid {
    double L[3];        // periodic edge (0 if open)
    double origin[3];   // lower corner used for binning
    double inv_cell[3]; // 1 / cell edge
    int nc[3];          // cells per axis
    int ncell;
    int periodic;
    int by_molecule;    // 1: "cell" = molecule, stencil = self (batched replicas)
    double edge[3];     // cell edge
    double inv_L[3];    // 1 / L (0 if open)
    int wrap[3];        // periodic axis with < 3 cells: per-pair minimum image also in the fp32 prefilter
    float Lf[3], inv_Lf[3];
};

// AEV constants in the form the kernels use (fp32, exp2-scaled).
struct AevConst {
    float rcr, rca;
    float pi_over_rcr, pi_over_rca;
    float eta_r_l2e;            // eta_r * log2(e)
    float eta_a_l2e;
    float eta_r, eta_a, zeta;
    float shf_r[NR], shf_a[DHP_MAX_SHF_A];
    float cos_z[DHP_MAX_SHF_Z], sin_z[DHP_MAX_SHF_Z];
    int n_a, n_z;               // angular grid: 8 x 4 (ANI-2x shape) or 4 x 8 (ANI-1x shape); n_a * n_z = 32
};

struct Weights {
    int n_models;
    float* blob;        // fp32 copy of the caller's blob (SIMT path)
    void* tc;           // tensor-path operand tiles (mlp_tc.cu), or nullptr
};

struct Profile {
    bool on;
    cudaEvent_t ev[64][DHP_N_PHASES + 1];
    int n_pending;
    int cur_slot;          // event row of the call being enqueued, or -1
    double ms[DHP_N_PHASES];
    int64_t calls;
};

// One captured hot call of a small system (api.cu): the kernels of such a call are 15-40 us each and the gaps between a dozen
// dependent launches are a sixth of the call, so the call is captured once per argument set and replayed as a CUDA graph.
struct GraphEntry {
    bool used;
    const void *pos, *species, *mol, *central, *weights, *E, *F;
    int64_t n, n_mol;
    float box[4];              // edges, [3] = 1 if periodic
    int mlp_mode;
    float skin;                // list reuse: the skin in force and which enqueue was captured (reuse check / forced rebuild)
    bool reuse_same;
    cudaGraphExec_t exec;      // null while the key has been seen only once (no graph yet)
    int64_t launches;          // kernels in the graph (dhp_launch_count)
    int64_t s_n_mol; bool s_periodic, s_partial, s_planes; int s_models;   // host-side state the enqueue leaves behind
    uint64_t stamp;
};
constexpr int N_GRAPHS = 8;

struct Ctx {
    cudaStream_t stream;
    dhp_params params;
    AevConst aevc;
    int64_t max_atoms, max_mols, max_rows, max_cells, pair_cap;
    int sm_count, cc_major;
    int mlp_mode;
    bool no_small_path;    // DHP_NO_SMALL_PATH=1 at dhp_create: small systems also take the general (cell list) path (tests)
    bool no_fwd_split;     // DHP_NO_FWD_SPLIT=1: small systems keep one warp per atom in the AEV forward pass (comparison)
    int tc_fuse;           // 1 (default): G1 runs inside the fused chain kernel (k_mlp_fused); DHP_TC_FUSE=0 keeps G1 + k_mlp_mid as two launches
    int tc_two;            // bit 0: G1, bit 1: B1 run with two row tiles per CTA sharing each weight K block (k_gemm_tc2) on large
                           // systems; DHP_TC_TWO=<bits> in the environment at dhp_create overrides the default (2: B1 only)
    int64_t launches;
    bool graph_on;         // small systems replay a captured graph (DHP_NO_GRAPH=1 at dhp_create turns it off)
    cudaStream_t cap_stream;   // the library's own stream for capture (the caller's may be the legacy default stream, which cannot capture)
    GraphEntry graphs[N_GRAPHS];
    uint64_t graph_clock;
    int64_t graph_replays;
    bool graph_large;      // systems above SMALL_N replay too (DHP_GRAPH_ALL=0 turns it off)
    bool graph_small;      // systems up to SMALL_N replay
    int64_t g_captures[2], g_replays[2];   // per size class (0 small, 1 large): graphs built and calls they served; a class whose
                           // graphs serve fewer than two calls each on average switches itself off (run_energy_forces)
    char cuda_err[256];
    Profile prof;

    // last call
    int64_t n_atoms, n_mol;
    int n_models;
    bool periodic;

    // workspace (device)
    unsigned* zero_arena;  // status, tc_sched, tile_mask, blk_sum, cell_count, cell_fill, e_atom, fsorted: zeroed by ONE memset per hot call
    size_t zero_words;
    int* ff_arena;         // row_slot, row_species: set to -1 by one memset per hot call
    Grid* grid;
    int* status;           // status word of the CURRENT hot call (in the zero arena)
    int* sticky;           // first fault since the last dhp_status(): survives the per-call memset, so a fault at an intermediate
                           // step of dhp_md_run (n calls, no host sync) is still reported
    int* cand_bad;         // device flag: a capacity fault truncated the candidate list - the next reuse call must rebuild
    unsigned* bbox;        // 6 ordered-uint min/max
    int* cell_of;          // [N] cell of caller's atom i
    int* perm_tmp;         // [N] cell-bucketed caller indices before the in-cell ordering
    int* cell_count;       // [max_cells+1]
    int* cell_start;       // [max_cells+1]
    int* cell_fill;        // [max_cells]
    int* perm;             // [N] sorted slot -> caller's index
    int* inv_perm;         // [N]
    float4* spos;          // [N] x,y,z, species bits
    int* smol;             // [N] molecule of sorted atom (0 if none)
    unsigned char* snc;    // [N] 1 = sorted atom is NOT a central atom of this call (partial evaluation), else 0
    bool partial;          // the last list was built with a central-atom mask
    // Verlet-skin reuse (dhp_set_skin): candidate pairs within rcr + skin of the positions of the last full build
    float skin;            // 0 = every call rebuilds from scratch
    unsigned* cand;        // [N][cand_stride] candidate entries: sorted slot | species << 28
    int* cand_cnt;         // [N]
    int cand_stride;
    float* pos_ref;        // [N][3] caller-order positions of the last full build
    int* rebuild;          // device flag of the current call: 1 = full build, 0 = candidate list reused
    bool cand_valid;       // host-side: a candidate list exists for (cand_n, cand_box, cand_mol, cand_nmol, cand_central)
    int64_t cand_n, cand_nmol;
    float cand_box[4];     // [3] = 1 if periodic
    const void* cand_mol;
    bool cand_central;
    int64_t n_rebuilds;    // full builds since dhp_set_skin (read back lazily: device counter)
    int* rebuild_count;    // device counter
    int* n_rad;            // [N]
    int* n_ang;            // [N]
    int* row_ptr;          // [N+1]
    int* col;              // [pair_cap] sorted-slot indices; each row ordered by (angular, radial-only) x species
    unsigned* tmp_col;     // [N][tmp_stride] unordered kept pairs of pass 1
    int tmp_stride;
    int* blk_sum;          // [N/256 + 2] pairs per 256-atom block
    int* blk_off;          // [N/256 + 2] exclusive scan, then total, then overflow flag
    unsigned short* seg_cnt; // [N][16] per row: angular count per species (0..6), n_ang (7), radial-only per species (8..14), (15)
    int* sp_count;         // [8]
    int* sp_start;         // [8] first row of each species group (multiple of ROW_TILE); [7] = end
    int* rowmap;           // [N] sorted slot -> row
    int* row_species;      // [max_rows] species of each row (-1 for padding rows)
    int* row_slot;         // [max_rows] sorted slot of each row (-1 for padding)
    int* blk_hist;         // [224 row keys][N/256 + 2] per-block histograms for the stable row assignment (key-major)
    int* rowkey_done;      // ticket counter of k_rowkey_scan's blocks (in the zero arena)
    int* key_start;        // [224] first row of each (species, feature-block class) key
    unsigned* amask;       // [N] feature blocks the atom's own AEV row can touch (bit b = 64-wide block b)
    unsigned* tile_mask;   // [max_rows / ROW_TILE] bit b: feature block b is non-zero for some row of the tile
    int* tc_sched;         // [8] dynamic tile counters of the tensor-path GEMMs
    int* col2feat;         // [AEV_LD] internal column -> canonical feature (-1: padding)
    float* aev;            // [max_rows][AEV_LD]  internal column order, see col2feat()
    float* grad;           // [max_rows][AEV_LD]  dE/dAEV
    float* e_atom;         // [max_rows]
    float* act[6];         // SIMT path intermediates: h1,h2,h3(delta3),delta2,delta1 ; see mlp_simt.cu (allocated on demand)
    int simt_models;       // networks per row those buffers hold (0 = not allocated)
    int max_models_seen;   // largest ensemble loaded on this context so far
    float* fsorted;        // [N][3] forces in sorted order
    double* e_out_tmp;     // [max(1,max_mols)]
    int* export_tmp;       // [N+1]
    // host-call staging
    float* st_pos; int* st_species; int* st_mol; double* st_E; float* st_F;
    void* tc_ws;           // tensor-path workspace (mlp_tc.cu)
    __half* aev_planes;    // [2][max_rows * AEV_LD] fp16 hi / lo planes of the AEV rows in the tiled layout of aev_tiled_off() (owned by tc_ws), or null
    bool aev_in_planes;    // the last forward pass wrote aev_planes (active blocks only) instead of aev
};

// ---- launch bookkeeping -------------------------------------------------------------------------
#define DHP_LAUNCH(ctx, kernel, grid, block, smem, ...)                         \
    do {                                                                        \
        kernel<<<(grid), (block), (smem), (ctx)->stream>>>(__VA_ARGS__);        \
        (ctx)->launches++;                                                      \
    } while (0)

int cuda_fail(Ctx* ctx, cudaError_t e, const char* what);
void prof_mark(Ctx* ctx, int boundary);   // records event `boundary` (start of phase `boundary`) of the current call when profiling
#define DHP_CUDA(ctx, call)                                            \
    do {                                                               \
        cudaError_t e__ = (call);                                      \
        if (e__ != cudaSuccess) return dhp::cuda_fail((ctx), e__, #call); \
    } while (0)

// ---- phases (each enqueues kernels on ctx->stream) ------------------------------------------------
bool nlist_reuse_same(const Ctx* ctx, int64_t n, const float* box_host, const int32_t* mol_offsets, int64_t n_mol, const uint8_t* central);
void nlist_reuse_mark(Ctx* ctx, int64_t n, const float* box_host, const int32_t* mol_offsets, int64_t n_mol, const uint8_t* central);
int nlist_build(Ctx* ctx, const float* pos, const float* box_host, const int32_t* species, int64_t n,
                const int32_t* mol_offsets, int64_t n_mol, const uint8_t* central = nullptr);
int nlist_export(Ctx* ctx, int32_t* row_ptr, int32_t* col, bool angular);
int aev_init(Ctx* ctx);                    // per-device kernel attributes
int aev_forward(Ctx* ctx, bool planes);   // planes: write the tensor path's fp16 hi/lo planes instead of fp32 rows
int aev_backward(Ctx* ctx, float* F_out);
int mlp_simt(Ctx* ctx, const Weights* w, bool forward_only);
int mlp_simt_ensure(Ctx* ctx, int n_models);   // setup-time (or first-use) sizing of the SIMT activations
void mlp_simt_free(Ctx* ctx);
int energy_reduce(Ctx* ctx, double* E_out);

// tensor path (mlp_tc.cu)
bool mlp_tc_available(Ctx* ctx);
int mlp_tc_alloc(Ctx* ctx);
int mlp_tc_ensure(Ctx* ctx, int n_models, bool layerwise);   // setup-time sizing of the tensor path's activation planes
void mlp_tc_free(Ctx* ctx);
int mlp_tc_weights(Ctx* ctx, Weights* w);
void mlp_tc_weights_free(Ctx* ctx, Weights* w);
int mlp_tc(Ctx* ctx, const Weights* w, bool forward_only);

// upper-triangle row-major index of the unordered species pair (canonical layout of the angular block, Q9)
__host__ __device__ inline int pairidx(int a, int b) {
    int u = a < b ? a : b, v = a < b ? b : a;
    return NSP * u - u * (u - 1) / 2 + (v - u);
}

// ---- internal column order of the AEV / dE/dAEV rows -------------------------------------------------
// The buffers are private to the library, so their column order is free.  Columns are arranged so that the
// 64-wide blocks a GEMM can skip are identically zero as often as possible for solvated biomolecules: species
// are ranked H, O, C, N, S, F, Cl ("priority" q), the angular blocks come first, ordered by (max q, min q) of
// the species pair - HH, HO, OO, HC, OC, CC, ... - then the radial blocks in priority order, then 16 zeros.
// A water-only tile touches 3 of the 16 blocks.  Debug exports and the weight preparation translate with
// col2feat(); the oracle and the tests only ever see the canonical order.
constexpr unsigned SP_PRIO_PACKED = 0x6541320u;   // nibble s: priority position of species s
constexpr unsigned PRIO_SP_PACKED = 0x6542130u;   // nibble q: species at priority position q
__host__ __device__ inline int sp_prio(int s) { return (int)((SP_PRIO_PACKED >> (4 * s)) & 7u); }
__host__ __device__ inline int prio_sp(int q) { return (int)((PRIO_SP_PACKED >> (4 * q)) & 7u); }
__host__ __device__ inline int ipair(int sa, int sb) {
    const int a = sp_prio(sa), b = sp_prio(sb);
    const int lo = a < b ? a : b, hi = a < b ? b : a;
    return hi * (hi + 1) / 2 + lo;
}
__host__ __device__ inline int rad_col(int s) { return AEV_ANG + NR * sp_prio(s); }
__host__ __device__ inline int col2feat(int c) {
    if (c < AEV_ANG) {
        const int ip = c >> 5, rem = c & 31;
        int hi = 0;
        while ((hi + 1) * (hi + 2) / 2 <= ip) ++hi;
        const int lo = ip - hi * (hi + 1) / 2;
        return AEV_RAD + 32 * pairidx(prio_sp(lo), prio_sp(hi)) + rem;
    }
    if (c < AEV_DIM) return NR * prio_sp((c - AEV_ANG) >> 4) + (c & 15);
    return -1;
}

}  // namespace dhp

struct dhp_nlist { dhp::Ctx* owner; };
struct dhp_ctx { dhp::Ctx c; dhp_nlist nl; };   // the opaque handles of include/dhp.h
