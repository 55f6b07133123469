/*
 * dhp.h — C ABI of libdhp.so: the ANI-2x-style neural-network potential of Deep-HP
 * (arXiv 2207.14276) as hand-written sm_100a CUDA.  One call evaluates the whole hot path
 *   neighbour search -> AEV (Eqs. 3-5) -> per-element MLP ensemble (Eq. 2) -> analytic forces.
 *
 * The interface restates the paper's own boundary (§2.2.1-2.2.2):
 *   - the MD engine stays the master and passes DEVICE addresses, no host copies (L128);
 *   - "provides positions and neighbor lists and gets energies and forces in return" (L130);
 *   - buffers are reserved once, proportional to N, never on the hot call (L134).
 *
 * Conventions
 *   - All functions return 0 (DHP_OK) or a negative DHP_E_* code; nothing throws or aborts.
 *   - "dev" pointers are CUDA device pointers valid on the device current at dhp_create();
 *     "host" pointers are ordinary host memory.  The caller owns every buffer it passes in.
 *   - The library owns the context, its workspace, neighbour lists and weight handles; they die with
 *     dhp_destroy().  A dhp_nlist is valid until the next dhp_nlist_build / dhp_ani_energy_forces
 *     on the same context.
 *   - Hot calls (dhp_nlist_build, dhp_ani_energy_forces) only enqueue work on the context's stream:
 *     no allocation, no host synchronisation.  Data-dependent faults (species outside 0..6, neighbour
 *     capacity overflow) set a device-side status word that stays set until dhp_status() reads it.
 *   - Units are the caller's: Å in, Hartree and Hartree/Å out (F = -dE/dr); no conversion inside.
 *   - Species index 0..6 = H, C, N, O, S, F, Cl.  The layout is fixed at compile time:
 *     16 radial shifts, 32 angular entries per species pair, AEV length 7*16 + 28*32 = 1008,
 *     networks 1008 -> 256 -> 192 -> 160 -> 1 with CELU (the published ANI-2x shape).  The angular grid is 8 x 4
 *     (ANI-2x) or 4 x 8 (ANI-1x / ANI-1ccx: species H, C, N, O = 0..3; its 384-entry AEV is the
 *     sub-vector of the 1008 layout that those four species span, and its narrower 384 -> 160 -> 128 -> 96 -> 1
 *     networks are loaded zero-padded into the fixed layout - same results, the cost of the wide shape).
 */
#ifndef DHP_H
#define DHP_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DHP_N_SPECIES 7
#define DHP_N_SHF_R 16
#define DHP_N_SHF_A 8    /* the ANI-2x angular grid: 8 radial shifts x 4 sections ... */
#define DHP_N_SHF_Z 4
#define DHP_MAX_SHF_A 8  /* ... capacity of the parameter arrays (ANI-1x grid: 4 x 8)  */
#define DHP_MAX_SHF_Z 8
#define DHP_AEV_DIM 1008
#define DHP_NET_PARAMS 338689 /* 1008*256+256 + 256*192+192 + 192*160+160 + 160+1 */

enum {
    DHP_OK = 0,
    DHP_E_BADARG = -1,   /* null pointer, negative size, n_models mismatch                       */
    DHP_E_CAPACITY = -2, /* n_atoms > max_atoms, n_mol > max_mols, or neighbour storage overflow  */
    DHP_E_BOX = -3,      /* a periodic edge is < 2*rc: the minimum image would not be unique      */
    DHP_E_SPECIES = -4,  /* a species index outside 0..6 (reported by dhp_status)                 */
    DHP_E_NOTIMPL = -5,
    DHP_E_CUDA = -6,     /* a CUDA runtime call failed; dhp_last_cuda_error() has the text        */
    DHP_E_NOMEM = -7
};

/* AEV hyper-parameters (Eqs. 3-5).  NULL in dhp_create = values of
 * the published ANI-2x model: Rcr 5.1, Rca 3.5, EtaR 19.7, EtaA 12.5, Zeta 14.1, CELU alpha 0.1,
 * ShfR = 0.8 + 0.2625 m, ShfA = 0.8 + 0.3375 a, ShfZ = (2k+1) pi/8. */
typedef struct dhp_params {
    float rcr;        /* radial cutoff R_c of Eq. 3 used in Eq. 4, Å          */
    float rca;        /* angular cutoff R_c of Eq. 3 used in Eq. 5, Å, <= rcr  */
    float eta_r;      /* eta of Eq. 4, Å^-2                                    */
    float eta_a;      /* eta of Eq. 5, Å^-2                                    */
    float zeta;       /* xi of Eq. 5                                           */
    float celu_alpha; /* CELU(x) = x (x>0), alpha (exp(x/alpha) - 1) otherwise */
    float shf_r[DHP_N_SHF_R];   /* R_s of Eq. 4, Å                                              */
    float shf_a[DHP_MAX_SHF_A]; /* R_s of Eq. 5, Å: the first n_shf_a entries                   */
    float shf_z[DHP_MAX_SHF_Z]; /* theta_s of Eq. 5: the first n_shf_z entries                  */
    int32_t n_shf_a;  /* angular grid of Eq. 5: 8 x 4 (ANI-2x shape) or 4 x 8 (ANI-1x / ANI-1ccx shape,                           */
    int32_t n_shf_z;  /* PAPER.md L87); n_shf_a * n_shf_z = 32 entries per species pair, laid out [a][z]                           */
} dhp_params;

typedef struct dhp_ctx dhp_ctx;         /* workspace sized for max_atoms, bound to one CUDA stream */
typedef struct dhp_nlist dhp_nlist;     /* device-resident CSR pair list, owned by the context     */
typedef struct dhp_weights dhp_weights; /* device-resident network parameters, owned by the context */

/* MLP arithmetic, dhp_set_mlp_mode().  AUTO, SIMT, TENSOR and TENSOR_LAYERWISE meet the parity tolerances against the
 * fp64 reference (energy within 1e-6 Hartree/atom, forces within 5e-5 Hartree/Å); TENSOR_FP16 is the opt-in
 * mixed-precision trade of PAPER.md L161 and does not. */
enum {
    DHP_MLP_AUTO = 0,   /* tensor path when available, else SIMT                                   */
    DHP_MLP_SIMT = 1,   /* fp32 FFMA GEMMs                                                          */
    DHP_MLP_TENSOR = 2, /* tcgen05 / TMEM GEMMs, fp16 two-term split operands (3 MMAs per product), fp32 accumulate.
                           One fused chain kernel runs every layer forward and the back-propagation down to the
                           first-layer deltas (AEV planes in, E_i and d1 out; h1, h2, h3 never leave the SM);
                           one more GEMM turns d1 into dE/dAEV                                                 */
    DHP_MLP_TENSOR_LAYERWISE = 3, /* same arithmetic, one launch per GEMM (bring-up / comparison path)  */
    DHP_MLP_TENSOR_FP16 = 4 /* the fused tensor path with ONE fp16 MMA per product (operands rounded to fp16, fp32
                               accumulate): the "mixed precision" option of PAPER.md L161.  Measured at 98 000 atoms with
                               8 networks: MLP phase 1.41 -> 1.16 ms; force errors 3-4e-4 Hartree/Å, i.e. outside the
                               5e-5 bar - never selected by AUTO                                                      */
};

/* Phases timed by dhp_profile_* (CUDA events on the context stream). */
enum {
    DHP_PHASE_NLIST = 0,   /* a1: binning, sort, CSR build                 */
    DHP_PHASE_AEV_FWD = 1, /* a2                                           */
    DHP_PHASE_MLP_G1 = 2,  /* a3: first layer, AEV -> h1 (all of a3 + a4 on the SIMT path)           */
    DHP_PHASE_MLP_MID = 3, /* a3 + a4: layers 2, 3, output, and their transposes, h1 -> (E_i, d1)    */
    DHP_PHASE_MLP_B1 = 4,  /* a4: first-layer transpose, d1 -> dE/dAEV; energy reduction             */
    DHP_PHASE_AEV_BWD = 5, /* a5 + force un-permutation                    */
    DHP_N_PHASES = 6
};

/* Create a context.  max_atoms / max_mols bound every later call (workspace is allocated here, once;
 * PAPER.md L134).  cuda_stream is a cudaStream_t (NULL = legacy default stream); all work of this
 * context is enqueued on it.  Errors: BADARG, NOMEM, CUDA. */
int dhp_create(dhp_ctx** out, const dhp_params* params, int64_t max_atoms, int64_t max_mols, void* cuda_stream);
int dhp_destroy(dhp_ctx* ctx);

/* Fixed limits of this build (compile-time constants of the kernels):
 *   n_models <= 8 (DHP_MAX_MODELS); at most 96 neighbours within rca and 192 within rcr of one atom (DHP_MAX_ANG,
 *   DHP_MAX_RAD: 3.4x / 3.5x the counts at 0.1 atoms/Å^3) - beyond that the call flags DHP_E_CAPACITY;
 *   total pair storage 160 directed pairs per atom of max_atoms. */
#define DHP_MAX_MODELS 8
#define DHP_MAX_ANG 96
#define DHP_MAX_RAD 192

/* Upload network parameters.  blob: HOST or DEVICE pointer to fp32, layout
 *   for e in 0..n_models-1: for s in 0..6: W1[256][1008], b1[256], W2[192][256], b2[192],
 *                                           W3[160][192], b3[160], W4[1][160], b4[1]
 * row-major [out][in]; n_floats must equal 338689*7*n_models.  The library keeps its own device copies
 * (fp32 for the SIMT path, split fp16 tiles for the tensor path); the caller may free blob afterwards.
 * Synchronises the stream (setup call, not a hot call).  Errors: BADARG, NOMEM, CUDA. */
int dhp_weights_load(dhp_ctx* ctx, const float* blob, int64_t n_floats, int n_models, dhp_weights** out);
int dhp_weights_free(dhp_ctx* ctx, dhp_weights* w);

/* a1 — neighbour search (linked-cell partition -> "pair list of indices").
 *   pos      dev fp32 [n_atoms][3], Å; may lie outside [0,L)
 *   box      HOST fp32 [3] cubic/orthorhombic periodic edges, or NULL for open boundaries
 *   species  dev int32 [n_atoms], 0..6
 *   mol_offsets dev int32 [n_mol+1] or NULL: atoms of molecule m are [mol_offsets[m], mol_offsets[m+1]);
 *            pairs never cross molecules (batched replicas); requires box == NULL
 *   rc       radial cutoff (must equal params.rcr); the angular sub-list radius is params.rca
 * A pair (i,j), i != j, is kept iff R^2 <= rc^2 with R^2 = (dx*dx + dy*dy) + dz*dz evaluated in fp64
 * without FMA contraction on the exactly converted fp32 inputs, d -= L*rint(d/L) per periodic axis
 * (Eq. 3's "R <= Rc").  The list is bit-exact, not approximately right.
 * Errors: BADARG, CAPACITY, BOX (host-side checks); SPECIES / CAPACITY via dhp_status(). */
int dhp_nlist_build(dhp_ctx* ctx, const float* pos, const float* box, const int32_t* species, int64_t n_atoms,
                    const int32_t* mol_offsets, int64_t n_mol, float rc, dhp_nlist** out);

/* Verlet-skin list reuse ("atomic positions do not move much between two time-steps").  skin > 0 (Å,
 * <= 4): a full build also records every pair within rc + skin; later calls on the same context with the same
 * n_atoms, box, mol_offsets pointer and masked/unmasked mode reuse the cell sort, the row assignment and that
 * candidate list for as long as no atom has moved more than skin/2 from the positions of the last full build (and
 * no atom changed species or central role) - checked on the device on every call, so a stale list is never used and
 * no host synchronisation is needed.  The list of every call is still exactly the canonical one (candidates are
 * filtered by the same fp64 predicate on the current positions).  skin = 0 (default) rebuilds on every call and
 * frees the candidate storage.  Setup call: allocates, synchronises.  Errors: BADARG, NOMEM. */
int dhp_set_skin(dhp_ctx* ctx, float skin);
/* Full builds since dhp_set_skin(skin > 0) (synchronises); every other hot call reused the candidate list. */
int64_t dhp_nlist_rebuild_count(dhp_ctx* ctx);

/* Number of directed pairs in the radial (<= rcr) and angular (<= rca) lists.  Synchronises.
 * (The counts are a call of their own because the caller needs them BEFORE it can allocate the col / col_ang buffers
 * that dhp_nlist_export fills.)
 * A dhp_nlist handle is a token of the context that built it: passing it to another context is DHP_E_BADARG. */
int dhp_nlist_sizes(dhp_ctx* ctx, const dhp_nlist* nl, int64_t* nnz, int64_t* nnz_ang);

/* Canonical form for parity: caller's atom numbering, both directions, each row ascending in j.
 * row_ptr / row_ptr_ang: dev int32 [n_atoms+1]; col / col_ang: dev int32 with room for nnz / nnz_ang
 * entries (dhp_nlist_sizes).  Any of the two (row_ptr, col) pairs may be NULL.  Not a hot call. */
int dhp_nlist_export(dhp_ctx* ctx, const dhp_nlist* nl, int32_t* row_ptr, int32_t* col,
                     int32_t* row_ptr_ang, int32_t* col_ang);

/* The hot call: a1..a5 in one go.  Builds its own pair list, then
 *   E  dev fp64 [max(1, n_mol)]  total energy (per molecule when mol_offsets is given), Hartree:
 *      E = (1/n_models) sum_e sum_i NN^{(e)}_{s_i}(G_i)            (Eq. 2; ensemble mean, L159)
 *   F  dev fp32 [n_atoms][3]     F = -dE/dr, Hartree/Å, caller's atom order
 * n_models must match the weight handle.  Asynchronous on the context stream. */
int dhp_ani_energy_forces(dhp_ctx* ctx, const float* pos, const float* box, const int32_t* species,
                          int64_t n_atoms, const int32_t* mol_offsets, int64_t n_mol,
                          const dhp_weights* weights, int n_models, double* E, float* F);

/* Energy only (a1, a2, a3): the same E as dhp_ani_energy_forces without the transpose-backward GEMMs (a4) and the
 * AEV backward (a5).  This is what reweighting needs: PAPER.md L228, BAR reweighting of existing trajectories uses
 * energies only and "avoids the costly computation of DNN gradients".  E as above; asynchronous. */
int dhp_ani_energy(dhp_ctx* ctx, const float* pos, const float* box, const int32_t* species, int64_t n_atoms,
                   const int32_t* mol_offsets, int64_t n_mol, const dhp_weights* weights, int n_models, double* E);

/* Partial evaluation over a subset of CENTRAL atoms - the building block of the multi-GPU decomposition.  The
 * energy is a sum of atomic terms over local environments (Eq. 2), which the paper shards by
 * spatial domains whose halo AEVs are recomputed redundantly (L134, L194: "~40 % loss").  Here a rank instead
 * evaluates only the atoms it owns as centres and no AEV is computed twice:
 *   central  dev uint8 [n_atoms], non-zero = atom i is a central atom of this call; NULL = all atoms
 *   E        E_c = (1/n_models) sum_e sum_{i central} NN^{(e)}_{s_i}(G_i)   (per molecule with mol_offsets)
 *   F        F_c = -dE_c/dr for ALL n_atoms atoms (a central atom's neighbours receive force from it)
 * Every atom still acts as a neighbour.  Over a partition of the atoms into central sets, the E_c and F_c add up
 * to the E and F of dhp_ani_energy_forces (up to fp32 summation order).  Asynchronous, like the full call. */
int dhp_ani_energy_forces_partial(dhp_ctx* ctx, const float* pos, const float* box, const int32_t* species,
                                  int64_t n_atoms, const int32_t* mol_offsets, int64_t n_mol,
                                  const dhp_weights* weights, int n_models, const uint8_t* central,
                                  double* E, float* F);

/* Multiple-timestep driver around the hot path (§2.4, Eqs. 8-9: the neural-network potential is
 * evaluated only at the OUTERMOST timestep; velocity Verlet, L144).  V_slow = the ANI potential of this library,
 * V_fast = harmonic bonds 1/2 k (r - r0)^2 - a stand-in for the bonded terms the paper keeps in the inner loop.
 * One outer step of length dt with n_inner inner steps d = dt / n_inner:
 *     v += (dt/2) a_slow ; [ v += (d/2) a_fast ; x += d v ; v += (d/2) a_fast ]^n_inner ; v += (dt/2) a_slow
 * (n_inner = 1 or n_bonds = 0: plain velocity Verlet with the total force).
 *   inv_mass  [n_atoms] acceleration per unit force, (Å/fs^2)/(Hartree/Å): 0.2625499639 / (mass in amu)
 *   bonds     int32 [n_bonds][2] atom pairs; bond_k Hartree/Å^2; bond_r0 Å    (host or device; copied at create)
 *   pos, vel  dev fp32 [n_atoms][3], Å and Å/fs, updated IN PLACE; positions are never re-wrapped into the box
 *   box, species, weights, n_models  as in dhp_ani_energy_forces (no mol_offsets: one system)
 *   E_out     dev fp64 [3] or NULL: E_ANI and E_bonds at the final positions, kinetic energy at the final velocities
 * dhp_md_run enqueues n_steps outer steps on the context stream without any host synchronisation; with
 * dhp_set_skin(skin > 0) the ANI calls reuse the neighbour list between outer steps.  The forces at the current
 * positions are carried from one run to the next; call dhp_md_reset after changing pos from outside. */
typedef struct dhp_md dhp_md;
int dhp_md_create(dhp_ctx* ctx, int64_t n_atoms, const float* inv_mass, const int32_t* bonds, const float* bond_k,
                  const float* bond_r0, int64_t n_bonds, dhp_md** out);
int dhp_md_destroy(dhp_ctx* ctx, dhp_md* md);
int dhp_md_reset(dhp_ctx* ctx, dhp_md* md);
int dhp_md_run(dhp_ctx* ctx, dhp_md* md, float* pos, float* vel, const float* box, const int32_t* species,
               const dhp_weights* weights, int n_models, float dt, int n_inner, int n_steps, double* E_out);

/* One outer step of the same scheme, split at the slow-force evaluation and restricted to the atoms [lo, hi) that a rank
 * OWNS - the building blocks of the multi-GPU MD loop (domain decomposition):
 *   dhp_md_open   v += (dt/2) a_slow ; [ v += (d/2) a_fast ; x += d v ; v += (d/2) a_fast ]^n_inner, WITHOUT the last fast
 *                 half kick                                                                          for atoms [lo, hi)
 *   ... the caller all-gathers the new positions, evaluates its partial slow force with
 *       dhp_ani_energy_forces_partial and reduce-scatters it (paper_2207_14276_b200/shard.py) ...
 *   dhp_md_close  v += (d/2) a_fast (the pending one, fast force at the final positions) + (dt/2) a_slow   for atoms [lo, hi)
 * After the pair the state is that of one full outer step.  BETWEEN the two calls the velocities lack that last fast half
 * kick (the two kicks are one kernel in dhp_md_close): do not read them there.  dhp_md_close must be given the dt and n_inner
 * of the dhp_md_open it completes, and there must be one - anything else is DHP_E_BADARG (an empty range [lo, lo) is a
 * no-op in both calls).
 * F_slow: dev fp32 [n_atoms][3], the TOTAL slow force; only rows [lo, hi) are read.  The md handle must have been
 * created with the bonds whose two atoms both lie in [lo, hi) (ranges are cut at molecule boundaries).  pos / vel are
 * the full [n_atoms][3] arrays; only rows [lo, hi) are written.  Asynchronous.  Errors: BADARG. */
int dhp_md_open(dhp_ctx* ctx, dhp_md* md, float* pos, float* vel, const float* box, const float* F_slow, float dt,
                int n_inner, int64_t lo, int64_t hi);
int dhp_md_close(dhp_ctx* ctx, dhp_md* md, float* vel, const float* F_slow, float dt, int n_inner, int64_t lo, int64_t hi);

/* Kinetic energy for callers that cannot allocate device memory.
 *
 * Who that is: a plug-in of an MD engine that claimed the whole GPU at start-up and hands out only the buffers it
 * registered (the set-up this library is written for: the engine is the master and reserves its memory once, PAPER.md
 * L128-134) - there a cudaMalloc may simply fail, and the engine's rules usually forbid it anyway; a per-step diagnostic
 * inside a running MD loop, where cudaMalloc / cudaFree would stall every stream of the device while they run; a process
 * whose framework allocator owns the device memory, so a raw cudaMalloc competes with it.  Every other call of this library
 * needs a dhp_ctx (dhp_create allocates the workspace) and, for the kinetic energy, a dhp_md handle (dhp_md_create
 * allocates the accumulators); this one needs neither and calls no cudaMalloc, cudaFree or allocating library routine,
 * on its first call or on any later one.
 *
 *   vel       dev fp32 [n_atoms][3], Å/fs
 *   inv_mass  dev fp32 [n_atoms], as in dhp_md_create: 0.2625499639 / (mass in amu)
 *   n_atoms   0 .. DHP_KINETIC_STATIC_MAX_ATOMS; more is refused with DHP_E_CAPACITY before anything is enqueued
 *             (n_atoms = 0 writes E_kin = 0)
 *   E_kin     dev fp64 [1], written (not added to): sum_i 1/2 |v_i|^2 / inv_mass_i, Hartree - the value dhp_md_run
 *             reports in E_out[2], up to the order of the fp64 additions (here fixed: block partials added in block order,
 *             so two calls on the same data give the same bits)
 *   cuda_stream  a cudaStream_t (NULL = legacy default stream) of the device that is CURRENT in the calling thread; the
 *             pointers must belong to that device.  Asynchronous: a memset of 256 bytes and one kernel are enqueued.
 *
 * Where the working memory lives instead: a fixed 33 KB array inside libdhp.so's device image (one partial sum per block of
 * 256 atoms, which is what sets the size limit, plus an arrival counter).  Every GPU that loads the library holds that array
 * until the process exits, whether this function is ever called or not.  Consequences a caller has to know:
 *   - there is ONE array per GPU, shared by every call from every thread and stream.  It keeps what the last call left; the
 *     function clears the counter itself at the start of each call.  Two calls that can run on the same GPU at the same
 *     time (different streams, or different host threads without ordering between their streams) race on it and both
 *     results are then undefined - order such calls yourself (same stream, or an event between the streams);
 *   - the first call on each device looks up the array's device address (cudaGetSymbolAddress, once per device, kept for
 *     later calls); that is set-up work, so make this first call before you start capturing any stream;
 * Errors: DHP_E_BADARG (null pointer with n_atoms > 0, null E_kin, n_atoms < 0), DHP_E_CAPACITY (n_atoms above the limit),
 * DHP_E_CUDA (the address lookup, the memset or the launch failed). */
#define DHP_KINETIC_STATIC_MAX_ATOMS 1048576
int dhp_kinetic_energy_static(const float* vel, const float* inv_mass, int64_t n_atoms, double* E_kin, void* cuda_stream);

/* Same computation with HOST buffers (pos, species, mol_offsets, E, F all host; pinned memory makes
 * the copies asynchronous): host->device copies, the kernels, device->host copies and one stream
 * synchronisation all happen inside the call.  This is the end-to-end entry point bench.py times. */
int dhp_ani_energy_forces_host(dhp_ctx* ctx, const float* pos, const float* box, const int32_t* species,
                               int64_t n_atoms, const int32_t* mol_offsets, int64_t n_mol,
                               const dhp_weights* weights, int n_models, double* E, float* F);

/* Synchronises the stream and returns the first data-dependent fault of ANY hot call since the previous dhp_status()
 * (DHP_E_SPECIES, DHP_E_CAPACITY), DHP_OK if there was none, or DHP_E_CUDA.  The word is sticky: every hot call folds its
 * own status into it on the device, so a fault at an intermediate call of an unsynchronised sequence (dhp_md_run
 * enqueues n_steps calls) is not lost; reading clears it.  After DHP_E_CAPACITY the results of the faulting call are
 * those of a truncated list (or of an empty one if the total pair storage overflowed); with list reuse the candidate
 * list is discarded and the next call rebuilds.  Within ONE call a capacity fault takes precedence over a species fault
 * (the word then reads DHP_E_CAPACITY whichever came first); across calls the first faulting call is the one reported. */
int dhp_status(dhp_ctx* ctx);

int dhp_set_mlp_mode(dhp_ctx* ctx, int mode);
/* 1 if this build and device can run the tcgen05 path (compute capability 10.x), else 0. */
int dhp_tensor_path_available(dhp_ctx* ctx);

/* Test-only exports, valid after a dhp_ani_energy_forces on the same context (synchronise):
 *   dhp_debug_aev            dev fp32 [n_atoms][1008]  G_i, caller's atom order, layout radial [s_j][m]
 *                            then angular [pairidx][a][z]
 *   dhp_debug_grad           dev fp32 [n_atoms][1008]  dE/dG_i (ensemble mean)
 *   dhp_debug_atomic_energy  dev fp32 [n_atoms]        E_i (ensemble mean) */
int dhp_debug_aev(dhp_ctx* ctx, float* aev);
int dhp_debug_grad(dhp_ctx* ctx, float* grad);
int dhp_debug_atomic_energy(dhp_ctx* ctx, float* e_atom);
/* Work accounting of the last call (host outputs, synchronises): the number of 128-row MLP tiles and the
 * total number of 64-wide feature blocks that are active over all tiles (at most 16 per tile).  The first
 * GEMM of the forward pass visits, and the last GEMM of the backward pass produces, only the active blocks
 * of a tile - the others are identically zero (absent neighbour species) - so the tensor-core work actually
 * issued for those two GEMMs is n_active_blocks / (16 n_row_tiles) of the dense count. */
int dhp_debug_tile_blocks(dhp_ctx* ctx, int64_t* n_row_tiles, int64_t* n_active_blocks);

/* Per-phase device timing.  dhp_profile_enable(ctx, 1) makes every hot call record CUDA events around
 * each phase on the context stream; dhp_profile_read synchronises and returns, for the calls since the
 * last dhp_profile_reset, the summed milliseconds per phase in ms[DHP_N_PHASES] and the call count. */
int dhp_profile_enable(dhp_ctx* ctx, int on);
int dhp_profile_reset(dhp_ctx* ctx);
int dhp_profile_read(dhp_ctx* ctx, double* ms, int64_t* n_calls);

/* Number of kernels this library has launched on the context since dhp_create (kernels of replayed graphs included). */
int64_t dhp_launch_count(dhp_ctx* ctx);
/* The hot call is captured once per argument set (pointers, sizes, box, mode, list-reuse state) into a CUDA graph and replayed
 * on later calls with the same arguments - same kernels, same results, no per-launch host work.  It matters most for small
 * systems (n_atoms <= 320: the solute of the hybrid scheme, the call RESPA's outer step makes, L200-208),
 * which are latency-bound; larger systems are replayed too (DHP_GRAPH_ALL=0 in the environment turns that off).  The graph is
 * built when an argument set is seen for the SECOND time; the first call with it runs as a plain enqueue, so a caller whose
 * arguments never repeat (new output buffers on every call, a new box each step) pays nothing for the mechanism.  Eight argument
 * sets are remembered per context (least recently used first out): rotate at most eight buffer sets, and pass the same E / F.
 * If graphs keep being built and then serve fewer than two calls each, the library stops building them for that size class.
 * Returns the number of hot calls served by a replay so far.  DHP_NO_GRAPH=1 in the environment at dhp_create turns the
 * mechanism off; it is also off while phase profiling is on. */
int64_t dhp_graph_replays(dhp_ctx* ctx);

const char* dhp_strerror(int code);
const char* dhp_last_cuda_error(dhp_ctx* ctx);
const char* dhp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DHP_H */
