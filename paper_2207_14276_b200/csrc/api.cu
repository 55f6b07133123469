// C ABI of libdhp.so (include/dhp.h): context / workspace, weight handles, the two hot calls.
#include <math.h>
#include <initializer_list>
#include <new>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "dhp_internal.cuh"
#if defined(__has_include)
#if __has_include("dhp_build_flags.h")
#include "dhp_build_flags.h"          // written by build.py: the extra compiler flags of this build
#endif
#endif
#ifndef DHP_EXTRA_FLAGS
#define DHP_EXTRA_FLAGS ""
#endif

namespace dhp {

int cuda_fail(Ctx* ctx, cudaError_t e, const char* what) {
    if (ctx) snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "%s: %s", what, cudaGetErrorString(e));
    return DHP_E_CUDA;
}

static void default_params(dhp_params* p) {
    p->rcr = 5.1f; p->rca = 3.5f; p->eta_r = 19.7f; p->eta_a = 12.5f; p->zeta = 14.1f; p->celu_alpha = 0.1f;
    for (int m = 0; m < NR; ++m) p->shf_r[m] = (float)(0.8 + 0.2625 * m);
    for (int a = 0; a < NA; ++a) p->shf_a[a] = (float)(0.8 + 0.3375 * a);
    for (int z = 0; z < NZ; ++z) p->shf_z[z] = (float)((2.0 * z + 1.0) * 3.14159265358979323846 / 8.0);
    for (int z = NZ; z < DHP_MAX_SHF_Z; ++z) p->shf_z[z] = 0.f;
    p->n_shf_a = NA; p->n_shf_z = NZ;
}

static void make_aev_const(const dhp_params& p, AevConst* k) {
    const double l2e = 1.4426950408889634074, pi = 3.14159265358979323846;
    k->rcr = p.rcr; k->rca = p.rca;
    k->pi_over_rcr = (float)(pi / (double)p.rcr); k->pi_over_rca = (float)(pi / (double)p.rca);
    k->eta_r_l2e = (float)((double)p.eta_r * l2e); k->eta_a_l2e = (float)((double)p.eta_a * l2e);
    k->eta_r = p.eta_r; k->eta_a = p.eta_a; k->zeta = p.zeta;
    for (int m = 0; m < NR; ++m) k->shf_r[m] = p.shf_r[m];
    k->n_a = p.n_shf_a; k->n_z = p.n_shf_z;
    for (int a = 0; a < DHP_MAX_SHF_A; ++a) k->shf_a[a] = a < p.n_shf_a ? p.shf_a[a] : 0.f;
    for (int z = 0; z < DHP_MAX_SHF_Z; ++z) {
        k->cos_z[z] = z < p.n_shf_z ? (float)cos((double)p.shf_z[z]) : 0.f;
        k->sin_z[z] = z < p.n_shf_z ? (float)sin((double)p.shf_z[z]) : 0.f;
    }
}

template <typename T>
static bool dalloc(T** p, size_t count) {
    *p = nullptr;
    return cudaMalloc((void**)p, sizeof(T) * (count ? count : 1)) == cudaSuccess;
}

static void graphs_invalidate(Ctx* ctx);
static void free_all(Ctx* c) {
    graphs_invalidate(c);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    void* ptrs[] = {c->sticky, c->cand_bad, c->grid, c->zero_arena, c->ff_arena, c->bbox, c->cell_of, c->perm_tmp, c->cell_start, c->perm,
                    c->inv_perm, c->spos, c->smol, c->snc, c->n_rad, c->n_ang, c->row_ptr, c->col, c->sp_count, c->sp_start,
                    c->rowmap, c->blk_hist, c->key_start, c->amask, c->col2feat, c->aev, c->grad,
                    c->e_out_tmp, c->export_tmp, c->cand, c->cand_cnt, c->pos_ref, c->rebuild, c->rebuild_count, c->tmp_col, c->blk_off, c->seg_cnt, c->st_pos, c->st_species, c->st_mol, c->st_E, c->st_F};
    for (void* p : ptrs) if (p) cudaFree(p);
    mlp_simt_free(c);
    mlp_tc_free(c);
    for (auto& row : c->prof.ev) for (auto& e : row) if (e) cudaEventDestroy(e);
}

static int check_args(Ctx* ctx, const float* pos, const float* box, const int32_t* species, int64_t n,
                      const int32_t* mol_offsets, int64_t n_mol) {
    if (!ctx || n < 0 || n_mol < 0) return DHP_E_BADARG;
    if (n > 0 && (!pos || !species)) return DHP_E_BADARG;
    if (n > ctx->max_atoms) return DHP_E_CAPACITY;
    if (mol_offsets && n_mol > 0) {
        if (box) return DHP_E_BADARG;
        if (n_mol > ctx->max_mols) return DHP_E_CAPACITY;
    }
    if (box)
        for (int c = 0; c < 3; ++c)
            if (!(box[c] >= 2.0f * ctx->params.rcr)) return DHP_E_BOX;
    return DHP_OK;
}

void prof_mark(Ctx* ctx, int boundary) {
    if (ctx->prof.on && ctx->prof.cur_slot >= 0) cudaEventRecord(ctx->prof.ev[ctx->prof.cur_slot][boundary], ctx->stream);
}

static void prof_drain(Ctx* ctx) {
    Profile& p = ctx->prof;
    if (p.n_pending == 0) return;
    cudaStreamSynchronize(ctx->stream);
    for (int s = 0; s < p.n_pending; ++s)
        for (int ph = 0; ph < DHP_N_PHASES; ++ph) {
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, p.ev[s][ph], p.ev[s][ph + 1]) == cudaSuccess) p.ms[ph] += ms;
        }
    p.calls += p.n_pending;
    p.n_pending = 0;
}

static int enqueue_energy_forces(Ctx* ctx, const float* pos, const float* box, const int32_t* species, int64_t n,
                                 const int32_t* mol_offsets, int64_t n_mol, const Weights* w, double* E, float* F,
                                 const uint8_t* central = nullptr) {
    ctx->prof.cur_slot = -1;
    if (ctx->prof.on) {
        if (ctx->prof.n_pending == 64) prof_drain(ctx);
        ctx->prof.cur_slot = ctx->prof.n_pending++;
    }
    int rc;
    prof_mark(ctx, DHP_PHASE_NLIST);
    if ((rc = nlist_build(ctx, pos, box, species, n, mol_offsets, n_mol, central)) != DHP_OK) return rc;
    prof_mark(ctx, DHP_PHASE_AEV_FWD);
    const bool tensor = ctx->mlp_mode == DHP_MLP_TENSOR || ctx->mlp_mode == DHP_MLP_TENSOR_LAYERWISE || ctx->mlp_mode == DHP_MLP_TENSOR_FP16 ||
                        (ctx->mlp_mode == DHP_MLP_AUTO && w->tc != nullptr);
    if (tensor && !w->tc) return DHP_E_NOTIMPL;
    if ((rc = aev_forward(ctx, tensor && ctx->aev_planes != nullptr)) != DHP_OK) return rc;
    prof_mark(ctx, DHP_PHASE_MLP_G1);
    const bool forward_only = F == nullptr;      // dhp_ani_energy: a1, a2, a3 only
    if (tensor) {
        rc = mlp_tc(ctx, w, forward_only);   // marks MLP_MID and MLP_B1 itself
    } else {
        rc = mlp_simt(ctx, w, forward_only);
        prof_mark(ctx, DHP_PHASE_MLP_MID);
        prof_mark(ctx, DHP_PHASE_MLP_B1);
    }
    if (rc != DHP_OK) return rc;
    if ((rc = energy_reduce(ctx, E)) != DHP_OK) return rc;
    prof_mark(ctx, DHP_PHASE_AEV_BWD);
    if (!forward_only && (rc = aev_backward(ctx, F)) != DHP_OK) return rc;
    prof_mark(ctx, DHP_N_PHASES);
    ctx->prof.cur_slot = -1;
    ctx->n_models = w->n_models;
    return DHP_OK;
}

static void graphs_invalidate(Ctx* ctx) {
    for (GraphEntry& g : ctx->graphs) {
        if (g.used && g.exec) cudaGraphExecDestroy(g.exec);
        g.used = false; g.exec = nullptr;
    }
}

// The hot call.  The enqueue of the kernels is captured ONCE per argument set (when that set is seen for the second time) into a
// CUDA graph on the library's own stream and replayed on the caller's stream afterwards - same kernels, same arithmetic, no per-launch host work and no gaps between
// dependent launches.  It matters most for small systems (n <= SMALL_N: the solute of the hybrid scheme, PAPER.md L112-118,
// L200-208 - the call RESPA's outer step makes: a dozen dependent 15-40 us launches); above SMALL_N it saves the ~1 % of the step
// that the nine short list kernels spend waiting for their launches, and switches itself off for a caller whose argument
// sets never repeat.  A changed pointer, size, box or mode is a
// new graph (8 keys are kept, least recently used first out).
static int run_energy_forces(Ctx* ctx, const float* pos, const float* box, const int32_t* species, int64_t n,
                             const int32_t* mol_offsets, int64_t n_mol, const Weights* w, double* E, float* F,
                             const uint8_t* central = nullptr) {
    {   // the SIMT scaffold's buffers exist from the first time it is going to run (never inside a graph capture)
        const bool tensor = ctx->mlp_mode >= DHP_MLP_TENSOR || (ctx->mlp_mode == DHP_MLP_AUTO && w->tc != nullptr);
        if (!tensor) { const int rc = mlp_simt_ensure(ctx, w->n_models); if (rc != DHP_OK) return rc; }
    }
    const bool large = n > SMALL_N;
    const bool small = ctx->graph_on && n > 0 && (large ? ctx->graph_large : ctx->graph_small) && !ctx->prof.on;
    // list reuse: the enqueue is one of two fixed sequences (device-side reuse check, or forced rebuild when the problem changed),
    // each with its own graph; the kernels of the path not taken are gated on the device as in a plain enqueue
    const bool skin_on = ctx->skin > 0.f && ctx->cand != nullptr && n > 0;
    const bool reuse_same = skin_on && nlist_reuse_same(ctx, n, box, mol_offsets, n_mol, central);
    const float skin_key = skin_on ? ctx->skin : 0.f;
    if (!small) return enqueue_energy_forces(ctx, pos, box, species, n, mol_offsets, n_mol, w, E, F, central);
    float bx[4] = {0.f, 0.f, 0.f, box ? 1.f : 0.f};
    if (box) for (int c = 0; c < 3; ++c) bx[c] = box[c];
    GraphEntry* hit = nullptr;
    GraphEntry* victim = &ctx->graphs[0];
    for (GraphEntry& g : ctx->graphs) {
        if (g.used && g.pos == pos && g.species == species && g.mol == mol_offsets && g.central == central && g.weights == w && g.E == E &&
            g.F == F && g.n == n && g.n_mol == n_mol && g.mlp_mode == ctx->mlp_mode && g.skin == skin_key && g.reuse_same == reuse_same &&
            memcmp(g.box, bx, sizeof(bx)) == 0) { hit = &g; break; }
        if (!g.used || (victim->used && g.stamp < victim->stamp)) victim = &g;
    }
    // A graph is built on the SECOND sighting of an argument set; the first sighting only records the key and runs as a plain
    // enqueue.  A caller whose arguments never repeat (fresh E / F buffers on every call, a new box per step, more rotating
    // position buffers than the table has entries) therefore never pays for a capture, at any system size.
    if (!hit) {
        if (victim->used && victim->exec) cudaGraphExecDestroy(victim->exec);
        victim->used = true; victim->exec = nullptr;
        victim->pos = pos; victim->species = species; victim->mol = mol_offsets; victim->central = central; victim->weights = w;
        victim->E = E; victim->F = F; victim->n = n; victim->n_mol = n_mol; victim->mlp_mode = ctx->mlp_mode;
        memcpy(victim->box, bx, sizeof(bx)); victim->skin = skin_key; victim->reuse_same = reuse_same;
        victim->stamp = ++ctx->graph_clock;
        return enqueue_energy_forces(ctx, pos, box, species, n, mol_offsets, n_mol, w, E, F, central);
    }
    if (!hit->exec) {
        // what is left to guard against is an argument set that comes back once or twice and then changes for good: when, after
        // 16 captures of a size class, the graphs have served fewer than two calls each on average, that class stops capturing
        int64_t& caps = ctx->g_captures[large ? 1 : 0];
        int64_t& reps = ctx->g_replays[large ? 1 : 0];
        if (caps >= 16 && reps < 2 * caps) {
            if (large) ctx->graph_large = false; else ctx->graph_small = false;
            return enqueue_energy_forces(ctx, pos, box, species, n, mol_offsets, n_mol, w, E, F, central);
        }
        ++caps;
        cudaStream_t user = ctx->stream;
        if (cudaStreamBeginCapture(ctx->cap_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
            cudaGetLastError();
            ctx->graph_on = false;                      // capture is not possible here: plain enqueue from now on
            return enqueue_energy_forces(ctx, pos, box, species, n, mol_offsets, n_mol, w, E, F, central);
        }
        ctx->stream = ctx->cap_stream;
        const int64_t l0 = ctx->launches;
        const int rc = enqueue_energy_forces(ctx, pos, box, species, n, mol_offsets, n_mol, w, E, F, central);
        ctx->stream = user;
        cudaGraph_t graph = nullptr;
        const cudaError_t e1 = cudaStreamEndCapture(ctx->cap_stream, &graph);
        if (rc != DHP_OK) { if (graph) cudaGraphDestroy(graph); cudaGetLastError(); return rc; }
        cudaGraphExec_t exec = nullptr;
        const cudaError_t e2 = e1 == cudaSuccess ? cudaGraphInstantiate(&exec, graph, 0) : e1;
        if (graph) cudaGraphDestroy(graph);
        if (e2 != cudaSuccess) {                          // could not build the graph: run the call the plain way
            cudaGetLastError();
            ctx->graph_on = false;
            ctx->launches = l0;
            return enqueue_energy_forces(ctx, pos, box, species, n, mol_offsets, n_mol, w, E, F, central);
        }
        hit->exec = exec;
        hit->launches = ctx->launches - l0;
        hit->s_n_mol = ctx->n_mol; hit->s_periodic = ctx->periodic; hit->s_partial = ctx->partial; hit->s_planes = ctx->aev_in_planes;
        hit->s_models = ctx->n_models;
        ctx->launches = l0;                               // counted per replay below
    }
    // the host-side state a plain enqueue would have left behind
    ctx->n_atoms = n; ctx->n_mol = hit->s_n_mol; ctx->periodic = hit->s_periodic; ctx->partial = hit->s_partial;
    ctx->aev_in_planes = hit->s_planes; ctx->n_models = hit->s_models;
    if (skin_on) nlist_reuse_mark(ctx, n, box, mol_offsets, n_mol, central); else ctx->cand_valid = false;
    hit->stamp = ++ctx->graph_clock;
    DHP_CUDA(ctx, cudaGraphLaunch(hit->exec, ctx->stream));
    ctx->launches += hit->launches;
    ctx->graph_replays++;
    ctx->g_replays[large ? 1 : 0]++;
    return DHP_OK;
}

// debug gathers: buffer rows -> caller's atom order
// With a column map the source is in the internal column order; feature blocks that are inactive for the row's
// tile were never computed (they are identically zero in the AEV and unused in dE/dAEV) and read as 0.
__global__ void k_gather_rows(const float* __restrict__ src, int ld_src, int ncol, const int* __restrict__ rowmap,
                              const int* __restrict__ inv_perm, int n, const int* __restrict__ col2feat,
                              const unsigned* __restrict__ tile_mask, float* __restrict__ dst) {
    int a = blockIdx.x;
    if (a >= n) return;
    const int row = rowmap[inv_perm[a]];
    if (row < 0) {                                   // not a central atom of the last (partial) call
        for (int c = threadIdx.x; c < ncol; c += blockDim.x) dst[(size_t)a * ncol + c] = 0.f;
        return;
    }
    const float* s = src + (size_t)row * ld_src;
    if (!col2feat) {
        for (int c = threadIdx.x; c < ncol; c += blockDim.x) dst[(size_t)a * ncol + c] = s[c];
        return;
    }
    const unsigned mask = tile_mask[row / ROW_TILE];
    for (int c = threadIdx.x; c < AEV_DIM; c += blockDim.x)
        dst[(size_t)a * ncol + col2feat[c]] = ((mask >> (c / KBLK)) & 1u) ? s[c] : 0.f;
}
// the same from the fp16 hi / lo planes the tensor path's forward pass writes (value = hi + lo)
__global__ void k_gather_planes(const __half* __restrict__ planes, size_t plane_stride, const int* __restrict__ rowmap,
                                const int* __restrict__ inv_perm, int n, const int* __restrict__ col2feat,
                                const unsigned* __restrict__ tile_mask, float* __restrict__ dst) {
    int a = blockIdx.x;
    if (a >= n) return;
    const int row = rowmap[inv_perm[a]];
    if (row < 0) {
        for (int c = threadIdx.x; c < AEV_DIM; c += blockDim.x) dst[(size_t)a * AEV_DIM + c] = 0.f;
        return;
    }
    const unsigned mask = tile_mask[row / ROW_TILE];
    for (int c = threadIdx.x; c < AEV_DIM; c += blockDim.x) {
        const size_t o = aev_tiled_off(row, c);
        dst[(size_t)a * AEV_DIM + col2feat[c]] = ((mask >> (c / KBLK)) & 1u) ? __half2float(planes[o]) + __half2float(planes[plane_stride + o]) : 0.f;
    }
}

}  // namespace dhp

using namespace dhp;

extern "C" {

struct dhp_weights { Weights w; };

int dhp_create(dhp_ctx** out, const dhp_params* params, int64_t max_atoms, int64_t max_mols, void* cuda_stream) {
    if (!out || max_atoms < 1 || max_mols < 0) return DHP_E_BADARG;
    *out = nullptr;
    dhp_ctx* h = new (std::nothrow) dhp_ctx();
    if (!h) return DHP_E_NOMEM;
    Ctx* c = &h->c;
    memset((void*)c, 0, sizeof(Ctx));
    c->stream = (cudaStream_t)cuda_stream;
    if (params) c->params = *params; else default_params(&c->params);
    if (!(c->params.rca > 0.f) || !(c->params.rcr >= c->params.rca) || !(c->params.celu_alpha > 0.f)) { delete h; return DHP_E_BADARG; }
    if (!((c->params.n_shf_a == 8 && c->params.n_shf_z == 4) || (c->params.n_shf_a == 4 && c->params.n_shf_z == 8))) { delete h; return DHP_E_BADARG; }
    make_aev_const(c->params, &c->aevc);
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) { delete h; return DHP_E_CUDA; }
    c->sm_count = prop.multiProcessorCount;
    { const char* e = getenv("DHP_NO_SMALL_PATH"); c->no_small_path = e && e[0] == '1'; }
    { const char* e = getenv("DHP_NO_GRAPH"); c->graph_on = !(e && e[0] == '1'); }
    { const char* e = getenv("DHP_GRAPH_ALL"); c->graph_large = !(e && e[0] == '0'); c->graph_small = true; c->g_captures[0] = c->g_captures[1] = c->g_replays[0] = c->g_replays[1] = 0; }
    if (c->graph_on && cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); c->graph_on = false; c->cap_stream = nullptr; }
    { const char* e = getenv("DHP_NO_FWD_SPLIT"); c->no_fwd_split = e && e[0] == '1'; }
    { const char* e = getenv("DHP_TC_FUSE"); c->tc_fuse = (e && e[0] == '0') ? 0 : 1; }
    { const char* e = getenv("DHP_TC_TWO"); c->tc_two = (e && e[0] >= '0' && e[0] <= '3') ? e[0] - '0' : 2; }   // two row tiles per CTA: B1 by default
    c->cc_major = prop.major;
    c->max_atoms = max_atoms;
    c->max_mols = max_mols;
    c->max_rows = (max_atoms + NSP * (ROW_ALIGN - 1) + ROW_ALIGN - 1) / ROW_ALIGN * ROW_ALIGN + ROW_ALIGN;
    c->max_cells = max_atoms * 2 > 256 ? max_atoms * 2 : 256;
    if (max_mols > c->max_cells) c->max_cells = max_mols;
    // neighbour storage: 160 directed pairs per atom on average (rho = 0.1 A^-3 gives 55 at 5.1 A); for tiny
    // systems every pair may be a neighbour
    c->pair_cap = max_atoms * 160;
    if (max_atoms < 161) c->pair_cap = max_atoms * (max_atoms - 1) + 1;
    // per-atom capacity of the pass-1 temporary rows (rho = 0.1 A^-3 gives 55 neighbours at 5.1 A)
    c->tmp_stride = (int)(max_atoms - 1 < 192 ? (max_atoms > 1 ? max_atoms - 1 : 1) : 192);
    const size_t N = (size_t)max_atoms, R = (size_t)c->max_rows, NC = (size_t)c->max_cells;
    const size_t NM = (size_t)(max_mols > 0 ? max_mols : 1);
    bool ok = true;
    ok &= dalloc(&c->grid, 1) && dalloc(&c->bbox, 8) && dalloc(&c->sticky, 1) && dalloc(&c->cand_bad, 1);
    ok &= dalloc(&c->cell_of, N) && dalloc(&c->perm_tmp, N) && dalloc(&c->cell_start, NC + 1);
    ok &= dalloc(&c->perm, N) && dalloc(&c->inv_perm, N) && dalloc(&c->spos, N) && dalloc(&c->smol, N) && dalloc(&c->snc, N);
    ok &= dalloc(&c->n_rad, N) && dalloc(&c->n_ang, N) && dalloc(&c->row_ptr, N + 1) && dalloc(&c->col, (size_t)c->pair_cap);
    ok &= dalloc(&c->tmp_col, N * c->tmp_stride) && dalloc(&c->blk_off, N / 64 + 3) && dalloc(&c->seg_cnt, N * 16);
    ok &= dalloc(&c->sp_count, 8) && dalloc(&c->sp_start, 8) && dalloc(&c->rowmap, N);
    ok &= dalloc(&c->blk_hist, (N / 256 + 2) * 224) && dalloc(&c->key_start, 224) && dalloc(&c->amask, N);
    ok &= dalloc(&c->aev, R * AEV_LD) && dalloc(&c->grad, R * AEV_LD);
    ok &= dalloc(&c->col2feat, AEV_LD);
    ok &= dalloc(&c->e_out_tmp, NM) && dalloc(&c->export_tmp, N + 1);
    {   // everything a hot call needs zeroed (or set to -1) lives in two arenas: two memsets per call instead of eleven
        size_t off = 0;
        auto take = [&](size_t words) { const size_t o = off; off += (words + 3) & ~(size_t)3; return o; };
        const size_t o_status = take(1), o_done = take(1), o_sched = take(8), o_tmask = take(R / ROW_TILE), o_bsum = take(N / 64 + 3), o_ccnt = take(NC + 1),
                     o_cfill = take(NC), o_eatom = take(R), o_fs = take(3 * N);
        c->zero_words = off;
        ok &= dalloc(&c->zero_arena, off) && dalloc(&c->ff_arena, 2 * R);
        if (ok) {
            c->status = (int*)c->zero_arena + o_status; c->rowkey_done = (int*)c->zero_arena + o_done; c->tc_sched = (int*)c->zero_arena + o_sched;
            c->tile_mask = (unsigned*)c->zero_arena + o_tmask; c->blk_sum = (int*)c->zero_arena + o_bsum;
            c->cell_count = (int*)c->zero_arena + o_ccnt; c->cell_fill = (int*)c->zero_arena + o_cfill;
            c->e_atom = (float*)c->zero_arena + o_eatom; c->fsorted = (float*)c->zero_arena + o_fs;
            c->row_slot = c->ff_arena; c->row_species = c->ff_arena + R;
        }
    }
    ok &= dalloc(&c->st_pos, 3 * N) && dalloc(&c->st_species, N) && dalloc(&c->st_mol, NM + 1) && dalloc(&c->st_E, NM) && dalloc(&c->st_F, 3 * N);
    if (ok) ok = aev_init(c) == DHP_OK;
    if (ok && mlp_tc_available(c)) ok = mlp_tc_alloc(c) == DHP_OK;
    if (ok) {
        for (auto& row : c->prof.ev) for (auto& e : row) ok &= cudaEventCreate(&e) == cudaSuccess;
        // padding rows are never written by the AEV kernel; keep them finite
        ok &= cudaMemset(c->aev, 0, sizeof(float) * R * AEV_LD) == cudaSuccess;
        ok &= cudaMemset(c->grad, 0, sizeof(float) * R * AEV_LD) == cudaSuccess;
        ok &= cudaMemset(c->status, 0, sizeof(int)) == cudaSuccess;
        ok &= cudaMemset(c->sticky, 0, sizeof(int)) == cudaSuccess && cudaMemset(c->cand_bad, 0, sizeof(int)) == cudaSuccess;
        int map[AEV_LD];
        for (int col = 0; col < AEV_LD; ++col) map[col] = col2feat(col);
        ok &= cudaMemcpy(c->col2feat, map, sizeof(map), cudaMemcpyHostToDevice) == cudaSuccess;
    }
    if (!ok) { cudaGetLastError(); free_all(c); delete h; return DHP_E_NOMEM; }
    *out = h;
    return DHP_OK;
}

int dhp_destroy(dhp_ctx* h) {
    if (!h) return DHP_E_BADARG;
    cudaStreamSynchronize(h->c.stream);
    free_all(&h->c);
    delete h;
    return DHP_OK;
}

int dhp_weights_load(dhp_ctx* h, const float* blob, int64_t n_floats, int n_models, dhp_weights** out) {
    if (!h || !blob || !out || n_models < 1 || n_models > MAX_MODELS) return DHP_E_BADARG;
    if (n_floats != (int64_t)NET_PARAMS * NSP * n_models) return DHP_E_BADARG;
    Ctx* c = &h->c;
    dhp_weights* w = new (std::nothrow) dhp_weights();
    if (!w) return DHP_E_NOMEM;
    w->w.n_models = n_models; w->w.blob = nullptr; w->w.tc = nullptr;
    if (cudaMalloc((void**)&w->w.blob, sizeof(float) * (size_t)n_floats) != cudaSuccess) { delete w; return DHP_E_NOMEM; }
    cudaError_t e = cudaMemcpyAsync(w->w.blob, blob, sizeof(float) * (size_t)n_floats, cudaMemcpyDefault, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) { cudaFree(w->w.blob); delete w; return cuda_fail(c, e, "weights upload"); }
    // activation workspaces are sized by the ensembles actually loaded (setup time; not by DHP_MAX_MODELS)
    if (n_models > c->max_models_seen) c->max_models_seen = n_models;
    {
        int rc = DHP_OK;
        const bool simt = c->mlp_mode == DHP_MLP_SIMT || !mlp_tc_available(c);
        if (simt) rc = mlp_simt_ensure(c, c->max_models_seen);
        if (rc == DHP_OK && mlp_tc_available(c)) rc = mlp_tc_ensure(c, c->max_models_seen, c->mlp_mode == DHP_MLP_TENSOR_LAYERWISE);
        if (rc != DHP_OK) { cudaFree(w->w.blob); delete w; return rc; }
        graphs_invalidate(c);                      // captured calls may hold the old buffers
    }
    if (mlp_tc_available(c)) {
        int rc = mlp_tc_weights(c, &w->w);
        if (rc != DHP_OK) { mlp_tc_weights_free(c, &w->w); cudaFree(w->w.blob); delete w; return rc; }
    }
    *out = w;
    return DHP_OK;
}

int dhp_weights_free(dhp_ctx* h, dhp_weights* w) {
    if (!h || !w) return DHP_E_BADARG;
    cudaStreamSynchronize(h->c.stream);
    graphs_invalidate(&h->c);                      // captured calls hold this handle's device pointers
    mlp_tc_weights_free(&h->c, &w->w);
    if (w->w.blob) cudaFree(w->w.blob);
    delete w;
    return DHP_OK;
}

int dhp_nlist_build(dhp_ctx* h, const float* pos, const float* box, const int32_t* species, int64_t n_atoms,
                    const int32_t* mol_offsets, int64_t n_mol, float rc, dhp_nlist** out) {
    if (!h) return DHP_E_BADARG;
    Ctx* c = &h->c;
    int r = check_args(c, pos, box, species, n_atoms, mol_offsets, n_mol);
    if (r != DHP_OK) return r;
    if (rc != c->params.rcr) return DHP_E_BADARG;
    r = nlist_build(c, pos, box, species, n_atoms, mol_offsets, n_mol);
    if (r != DHP_OK) return r;
    if (out) { h->nl.owner = c; *out = &h->nl; }     // the list lives in the context workspace; the handle is a per-context token
    return DHP_OK;
}

int dhp_nlist_sizes(dhp_ctx* h, const dhp_nlist* nl, int64_t* nnz, int64_t* nnz_ang) {
    if (!h || !nl || nl->owner != &h->c) return DHP_E_BADARG;      // a list handle belongs to the context that built it
    Ctx* c = &h->c;
    const int n = (int)c->n_atoms;
    int total = 0;
    DHP_CUDA(c, cudaMemcpyAsync(&total, c->row_ptr + n, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    DHP_CUDA(c, cudaStreamSynchronize(c->stream));
    if (nnz) *nnz = total;
    if (nnz_ang) {
        int64_t t = 0;
        if (n > 0) {
            int* tmp = (int*)malloc(sizeof(int) * n);
            if (!tmp) return DHP_E_NOMEM;
            cudaError_t e = cudaMemcpy(tmp, c->n_ang, sizeof(int) * n, cudaMemcpyDeviceToHost);
            if (e != cudaSuccess) { free(tmp); return cuda_fail(c, e, "n_ang download"); }
            for (int i = 0; i < n; ++i) t += tmp[i];
            free(tmp);
        }
        *nnz_ang = t;
    }
    return DHP_OK;
}

int dhp_nlist_export(dhp_ctx* h, const dhp_nlist* nl, int32_t* row_ptr, int32_t* col, int32_t* row_ptr_ang, int32_t* col_ang) {
    if (!h || !nl || nl->owner != &h->c) return DHP_E_BADARG;
    Ctx* c = &h->c;
    int r = DHP_OK;
    if (row_ptr) r = nlist_export(c, row_ptr, col, false);
    if (r == DHP_OK && row_ptr_ang) r = nlist_export(c, row_ptr_ang, col_ang, true);
    return r;
}

int dhp_ani_energy_forces(dhp_ctx* h, const float* pos, const float* box, const int32_t* species, int64_t n_atoms,
                          const int32_t* mol_offsets, int64_t n_mol, const dhp_weights* weights, int n_models,
                          double* E, float* F) {
    if (!h || !weights || !E || (n_atoms > 0 && !F)) return DHP_E_BADARG;
    Ctx* c = &h->c;
    if (n_models != weights->w.n_models) return DHP_E_BADARG;
    int r = check_args(c, pos, box, species, n_atoms, mol_offsets, n_mol);
    if (r != DHP_OK) return r;
    return run_energy_forces(c, pos, box, species, n_atoms, mol_offsets, n_mol, &weights->w, E, F);
}

int dhp_ani_energy_forces_partial(dhp_ctx* h, const float* pos, const float* box, const int32_t* species, int64_t n_atoms,
                                  const int32_t* mol_offsets, int64_t n_mol, const dhp_weights* weights, int n_models,
                                  const uint8_t* central, double* E, float* F) {
    if (!h || !weights || !E || (n_atoms > 0 && !F)) return DHP_E_BADARG;
    Ctx* c = &h->c;
    if (n_models != weights->w.n_models) return DHP_E_BADARG;
    int r = check_args(c, pos, box, species, n_atoms, mol_offsets, n_mol);
    if (r != DHP_OK) return r;
    return run_energy_forces(c, pos, box, species, n_atoms, mol_offsets, n_mol, &weights->w, E, F, central);
}

int dhp_ani_energy(dhp_ctx* h, const float* pos, const float* box, const int32_t* species, int64_t n_atoms,
                   const int32_t* mol_offsets, int64_t n_mol, const dhp_weights* weights, int n_models, double* E) {
    if (!h || !weights || !E) return DHP_E_BADARG;
    Ctx* c = &h->c;
    if (n_models != weights->w.n_models) return DHP_E_BADARG;
    int r = check_args(c, pos, box, species, n_atoms, mol_offsets, n_mol);
    if (r != DHP_OK) return r;
    return run_energy_forces(c, pos, box, species, n_atoms, mol_offsets, n_mol, &weights->w, E, nullptr);
}

int dhp_ani_energy_forces_host(dhp_ctx* h, const float* pos, const float* box, const int32_t* species, int64_t n_atoms,
                               const int32_t* mol_offsets, int64_t n_mol, const dhp_weights* weights, int n_models,
                               double* E, float* F) {
    if (!h || !weights || !E || (n_atoms > 0 && !F)) return DHP_E_BADARG;
    Ctx* c = &h->c;
    if (n_models != weights->w.n_models) return DHP_E_BADARG;
    int r = check_args(c, pos, box, species, n_atoms, mol_offsets, n_mol);
    if (r != DHP_OK) return r;
    const bool by_mol = mol_offsets && n_mol > 0;
    const int64_t ne = by_mol ? n_mol : 1;
    cudaStream_t st = c->stream;
    if (n_atoms > 0) {
        DHP_CUDA(c, cudaMemcpyAsync(c->st_pos, pos, sizeof(float) * 3 * n_atoms, cudaMemcpyHostToDevice, st));
        DHP_CUDA(c, cudaMemcpyAsync(c->st_species, species, sizeof(int) * n_atoms, cudaMemcpyHostToDevice, st));
    }
    if (by_mol) DHP_CUDA(c, cudaMemcpyAsync(c->st_mol, mol_offsets, sizeof(int) * (n_mol + 1), cudaMemcpyHostToDevice, st));
    r = run_energy_forces(c, c->st_pos, box, c->st_species, n_atoms, by_mol ? c->st_mol : nullptr, n_mol, &weights->w, c->st_E, c->st_F);
    if (r != DHP_OK) return r;
    DHP_CUDA(c, cudaMemcpyAsync(E, c->st_E, sizeof(double) * ne, cudaMemcpyDeviceToHost, st));
    if (n_atoms > 0) DHP_CUDA(c, cudaMemcpyAsync(F, c->st_F, sizeof(float) * 3 * n_atoms, cudaMemcpyDeviceToHost, st));
    DHP_CUDA(c, cudaStreamSynchronize(st));
    return DHP_OK;
}

int dhp_status(dhp_ctx* h) {
    if (!h) return DHP_E_BADARG;
    Ctx* c = &h->c;
    // the sticky word holds the first fault of any hot call since the last dhp_status(); the per-call word covers calls
    // that end before the fold (dhp_nlist_build alone)
    int s = 0, sticky = 0;
    cudaError_t e = cudaMemcpyAsync(&s, c->status, sizeof(int), cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(&sticky, c->sticky, sizeof(int), cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->sticky, 0, sizeof(int), c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->status, 0, sizeof(int), c->stream);   // reading clears both words: a fault of the LAST call is reported once
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "status");
    return sticky != 0 ? sticky : s;
}

int dhp_set_mlp_mode(dhp_ctx* h, int mode) {
    if (!h || mode < DHP_MLP_AUTO || mode > DHP_MLP_TENSOR_FP16) return DHP_E_BADARG;
    if (mode >= DHP_MLP_TENSOR && !mlp_tc_available(&h->c)) return DHP_E_NOTIMPL;
    h->c.mlp_mode = mode;
    if (h->c.max_models_seen > 0) {               // the workspaces of the newly selected path (setup call: may allocate)
        int rc = DHP_OK;
        if (mode == DHP_MLP_SIMT) rc = mlp_simt_ensure(&h->c, h->c.max_models_seen);
        else rc = mlp_tc_ensure(&h->c, h->c.max_models_seen, mode == DHP_MLP_TENSOR_LAYERWISE);
        if (rc != DHP_OK) return rc;
        graphs_invalidate(&h->c);
    }
    return DHP_OK;     // (captured graphs are keyed on the mode)
}

int dhp_set_skin(dhp_ctx* h, float skin) {
    if (!h || !(skin >= 0.f) || skin > 4.0f) return DHP_E_BADARG;
    Ctx* c = &h->c;
    cudaStreamSynchronize(c->stream);
    graphs_invalidate(c);                          // captured calls hold the candidate buffers of the old skin (or none)
    for (void* p : {(void*)c->cand, (void*)c->cand_cnt, (void*)c->pos_ref, (void*)c->rebuild, (void*)c->rebuild_count}) if (p) cudaFree(p);
    c->cand = nullptr; c->cand_cnt = nullptr; c->pos_ref = nullptr; c->rebuild = nullptr; c->rebuild_count = nullptr;
    c->skin = 0.f; c->cand_valid = false; c->cand_stride = 0;
    if (skin == 0.f) return DHP_OK;
    // candidate rows scale with the list volume: tmp_stride x ((rcr + skin) / rcr)^3, in whole warps
    const double f = ((double)c->params.rcr + skin) / (double)c->params.rcr;
    int64_t stride = ((int64_t)ceil(c->tmp_stride * f * f * f) + 31) / 32 * 32;
    if (stride > c->max_atoms - 1) stride = c->max_atoms > 1 ? c->max_atoms - 1 : 1;
    const size_t N = (size_t)c->max_atoms;
    bool ok = dalloc(&c->cand, N * (size_t)stride) && dalloc(&c->cand_cnt, N) && dalloc(&c->pos_ref, 3 * N) && dalloc(&c->rebuild, 1) &&
              dalloc(&c->rebuild_count, 1);
    if (ok) ok = cudaMemset(c->rebuild_count, 0, sizeof(int)) == cudaSuccess;
    if (!ok) {
        cudaGetLastError();
        for (void* p : {(void*)c->cand, (void*)c->cand_cnt, (void*)c->pos_ref, (void*)c->rebuild, (void*)c->rebuild_count}) if (p) cudaFree(p);
        c->cand = nullptr; c->cand_cnt = nullptr; c->pos_ref = nullptr; c->rebuild = nullptr; c->rebuild_count = nullptr;
        return DHP_E_NOMEM;
    }
    c->cand_stride = (int)stride;
    c->skin = skin;
    return DHP_OK;
}

int64_t dhp_nlist_rebuild_count(dhp_ctx* h) {
    if (!h || !h->c.rebuild_count) return 0;
    int v = 0;
    if (cudaMemcpyAsync(&v, h->c.rebuild_count, sizeof(int), cudaMemcpyDeviceToHost, h->c.stream) != cudaSuccess) return -1;
    if (cudaStreamSynchronize(h->c.stream) != cudaSuccess) return -1;
    return v;
}

int dhp_tensor_path_available(dhp_ctx* h) { return h && mlp_tc_available(&h->c) ? 1 : 0; }

static int debug_gather(dhp_ctx* h, const float* src, int ld, int ncol, float* dst, bool feature_rows) {
    if (!h || !dst) return DHP_E_BADARG;
    Ctx* c = &h->c;
    const int n = (int)c->n_atoms;
    if (n == 0) return DHP_OK;
    DHP_LAUNCH(c, k_gather_rows, n, 128, 0, src, ld, ncol, c->rowmap, c->inv_perm, n,
               feature_rows ? c->col2feat : (const int*)nullptr, c->tile_mask, dst);
    DHP_CUDA(c, cudaGetLastError());
    DHP_CUDA(c, cudaStreamSynchronize(c->stream));
    return DHP_OK;
}
int dhp_debug_aev(dhp_ctx* h, float* aev) {
    if (!h || !aev) return DHP_E_BADARG;
    Ctx* c = &h->c;
    if (!c->aev_in_planes) return debug_gather(h, c->aev, AEV_LD, AEV_DIM, aev, true);
    const int n = (int)c->n_atoms;
    if (n == 0) return DHP_OK;
    DHP_LAUNCH(c, k_gather_planes, n, 128, 0, c->aev_planes, (size_t)c->max_rows * AEV_LD, c->rowmap, c->inv_perm, n, c->col2feat,
               c->tile_mask, aev);
    DHP_CUDA(c, cudaGetLastError());
    DHP_CUDA(c, cudaStreamSynchronize(c->stream));
    return DHP_OK;
}
int dhp_debug_grad(dhp_ctx* h, float* grad) { return h ? debug_gather(h, h->c.grad, AEV_LD, AEV_DIM, grad, true) : DHP_E_BADARG; }
int dhp_debug_atomic_energy(dhp_ctx* h, float* e) { return h ? debug_gather(h, h->c.e_atom, 1, 1, e, false) : DHP_E_BADARG; }

int dhp_debug_tile_blocks(dhp_ctx* h, int64_t* n_row_tiles, int64_t* n_active_blocks) {
    if (!h || !n_row_tiles || !n_active_blocks) return DHP_E_BADARG;
    Ctx* c = &h->c;
    *n_row_tiles = 0; *n_active_blocks = 0;
    if (c->n_atoms == 0) return DHP_OK;
    int sp_start[8];
    DHP_CUDA(c, cudaMemcpyAsync(sp_start, c->sp_start, sizeof(sp_start), cudaMemcpyDeviceToHost, c->stream));
    DHP_CUDA(c, cudaStreamSynchronize(c->stream));
    const int nt = sp_start[NSP] / ROW_TILE;
    unsigned* m = (unsigned*)malloc(sizeof(unsigned) * (nt > 0 ? nt : 1));
    if (!m) return DHP_E_NOMEM;
    cudaError_t e = cudaMemcpy(m, c->tile_mask, sizeof(unsigned) * nt, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) { free(m); return cuda_fail(c, e, "tile mask download"); }
    int64_t blocks = 0;
    for (int t = 0; t < nt; ++t) blocks += __builtin_popcount(m[t] ? m[t] : (1u << 14));   // an all-zero tile runs one block
    free(m);
    *n_row_tiles = nt; *n_active_blocks = blocks;
    return DHP_OK;
}

int dhp_profile_enable(dhp_ctx* h, int on) {
    if (!h) return DHP_E_BADARG;
    prof_drain(&h->c);
    h->c.prof.on = on != 0;
    return DHP_OK;
}
int dhp_profile_reset(dhp_ctx* h) {
    if (!h) return DHP_E_BADARG;
    prof_drain(&h->c);
    for (double& m : h->c.prof.ms) m = 0.0;
    h->c.prof.calls = 0;
    return DHP_OK;
}
int dhp_profile_read(dhp_ctx* h, double* ms, int64_t* n_calls) {
    if (!h || !ms) return DHP_E_BADARG;
    prof_drain(&h->c);
    for (int p = 0; p < DHP_N_PHASES; ++p) ms[p] = h->c.prof.ms[p];
    if (n_calls) *n_calls = h->c.prof.calls;
    return DHP_OK;
}

int64_t dhp_launch_count(dhp_ctx* h) { return h ? h->c.launches : 0; }
int64_t dhp_graph_replays(dhp_ctx* h) { return h ? h->c.graph_replays : 0; }

const char* dhp_strerror(int code) {
    switch (code) {
        case DHP_OK: return "ok";
        case DHP_E_BADARG: return "bad argument";
        case DHP_E_CAPACITY: return "capacity exceeded (atoms, molecules or neighbour storage)";
        case DHP_E_BOX: return "periodic box edge shorter than twice the radial cutoff";
        case DHP_E_SPECIES: return "species index outside 0..6";
        case DHP_E_NOTIMPL: return "not implemented / not available on this device";
        case DHP_E_CUDA: return "CUDA runtime error";
        case DHP_E_NOMEM: return "out of memory";
        default: return "unknown error";
    }
}
const char* dhp_last_cuda_error(dhp_ctx* h) { return h ? h->c.cuda_err : ""; }
// "dhp 0.1 (sm_100a)" for a default build; a build with extra compiler flags (DHP_NVCC_EXTRA: the timing-experiment macros, some of
// which give wrong results by design) says so: "dhp 0.1 (sm_100a) [extra flags: ...]" - binding.load_library() refuses such a library
const char* dhp_version(void) { return sizeof(DHP_EXTRA_FLAGS) > 1 ? "dhp 0.1 (sm_100a) [extra flags: " DHP_EXTRA_FLAGS "]" : "dhp 0.1 (sm_100a)"; }

}  // extern "C"
