// f1 — multiple-timestep driver around the hot path (§2.4, Eqs. 8-9; velocity Verlet L144).
//
// The paper's RESPA split evaluates the neural-network potential only at the OUTERMOST timestep and keeps cheap
// bonded terms in the inner loop.  Here: V_slow = the ANI potential (dhp_ani_energy_forces, a1..a5), V_fast =
// harmonic bonds 1/2 k (r - r0)^2 (a stand-in for the bonded terms; AMOEBA is out of scope).  One outer step of
// length dt with n inner steps of length d = dt / n is the symmetric factorisation
//     v += (dt/2) a_slow ; [ v += (d/2) a_fast ; x += d v ; v += (d/2) a_fast ]^n ; v += (dt/2) a_slow
// which for n = 1 (or no bonds) is plain velocity Verlet with the total force.  Everything is enqueued on the
// context's stream; there is no host synchronisation inside a run, and with dhp_set_skin the neighbour list of
// the ANI call is reused between outer steps ("atomic positions do not move much between two time-steps", L134).
#include <initializer_list>
#include <mutex>
#include <new>
#include <string.h>

#include "dhp_internal.cuh"

namespace dhp {

struct Md {
    int64_t n_atoms, n_bonds;
    float* inv_mass;   // [N]  (Å/fs^2) per (Hartree/Å): acceleration = inv_mass * force
    int* bonds;        // [n_bonds][2]
    float* bond_k;     // [n_bonds] Hartree/Å^2
    float* bond_r0;    // [n_bonds] Å
    float* f_slow;     // [N][3]
    float* f_fast;     // [N][3]
    double* e;         // [3] E_slow, E_fast, E_kin
    bool primed;       // f_slow / f_fast hold the forces at the current positions
    float open_dt;     // dhp_md_open .. dhp_md_close: the step in flight (0 = none): close must finish the step open began
    int open_n_inner;
};

// v += inv_m (ca Fa + cb Fb); optionally x += delta v
__global__ void k_md_kick_drift(float* __restrict__ pos, float* __restrict__ vel, const float* __restrict__ inv_mass,
                                const float* __restrict__ Fa, float ca, const float* __restrict__ Fb, float cb, float delta,
                                int n3, int t0 = 0) {
    const int t = t0 + blockIdx.x * blockDim.x + threadIdx.x;      // components [t0, n3): all atoms, or the range a rank owns
    if (t >= n3) return;
    float f = 0.f;
    if (Fa) f = ca * Fa[t];
    if (Fb) f = fmaf(cb, Fb[t], f);
    const float v = fmaf(inv_mass[t / 3], f, vel[t]);
    vel[t] = v;
    if (delta != 0.f) pos[t] = fmaf(delta, v, pos[t]);
}

// harmonic bonds: E = sum 1/2 k (r - r0)^2, F = -dE/dr (minimum image in a periodic box)
__global__ void k_md_bonds(const float* __restrict__ pos, float Lx, float Ly, float Lz, int periodic, const int* __restrict__ bonds,
                           const float* __restrict__ bond_k, const float* __restrict__ bond_r0, int n_bonds, float* __restrict__ F,
                           double* __restrict__ E) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    double e = 0.0;
    if (b < n_bonds) {
        const int i = bonds[2 * b], j = bonds[2 * b + 1];
        float dx = pos[3 * j] - pos[3 * i], dy = pos[3 * j + 1] - pos[3 * i + 1], dz = pos[3 * j + 2] - pos[3 * i + 2];
        if (periodic) {
            dx -= Lx * rintf(dx / Lx); dy -= Ly * rintf(dy / Ly); dz -= Lz * rintf(dz / Lz);
        }
        const float r = sqrtf(dx * dx + dy * dy + dz * dz);
        const float dr = r - bond_r0[b], k = bond_k[b];
        e = 0.5 * (double)k * (double)dr * (double)dr;
        const float s = r > 0.f ? k * dr / r : 0.f;          // force on i is +s d, on j is -s d
        atomicAdd(&F[3 * i], s * dx); atomicAdd(&F[3 * i + 1], s * dy); atomicAdd(&F[3 * i + 2], s * dz);
        atomicAdd(&F[3 * j], -s * dx); atomicAdd(&F[3 * j + 1], -s * dy); atomicAdd(&F[3 * j + 2], -s * dz);
    }
    for (int o = 16; o; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
    if ((threadIdx.x & 31) == 0 && e != 0.0) atomicAdd(E, e);
}

// E_kin = sum 1/2 v^2 / inv_mass
__global__ void k_md_kinetic(const float* __restrict__ vel, const float* __restrict__ inv_mass, int n, double* __restrict__ E) {
    double e = 0.0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const double vx = vel[3 * i], vy = vel[3 * i + 1], vz = vel[3 * i + 2];
        e += 0.5 * (vx * vx + vy * vy + vz * vz) / (double)inv_mass[i];
    }
    for (int o = 16; o; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
    if ((threadIdx.x & 31) == 0) atomicAdd(E, e);
}

static int fast_forces(Ctx* c, Md* m, const float* pos, const float* box) {
    if (m->n_bonds == 0) return DHP_OK;
    DHP_CUDA(c, cudaMemsetAsync(m->f_fast, 0, sizeof(float) * 3 * m->n_atoms, c->stream));
    DHP_CUDA(c, cudaMemsetAsync(m->e + 1, 0, sizeof(double), c->stream));
    DHP_LAUNCH(c, k_md_bonds, (int)((m->n_bonds + 127) / 128), 128, 0, pos, box ? box[0] : 0.f, box ? box[1] : 0.f, box ? box[2] : 0.f,
               box ? 1 : 0, m->bonds, m->bond_k, m->bond_r0, (int)m->n_bonds, m->f_fast, m->e + 1);
    return DHP_OK;
}

}  // namespace dhp

using namespace dhp;

// the hot call of api.cu
extern "C" int dhp_ani_energy_forces(dhp_ctx* ctx, const float* pos, const float* box, const int32_t* species, int64_t n_atoms,
                                     const int32_t* mol_offsets, int64_t n_mol, const dhp_weights* weights, int n_models,
                                     double* E, float* F);
struct dhp_md { Md m; };

extern "C" {

int dhp_md_create(dhp_ctx* h, int64_t n_atoms, const float* inv_mass, const int32_t* bonds, const float* bond_k,
                  const float* bond_r0, int64_t n_bonds, dhp_md** out) {
    if (!h || !out || n_atoms < 1 || !inv_mass || n_bonds < 0 || (n_bonds > 0 && (!bonds || !bond_k || !bond_r0))) return DHP_E_BADARG;
    Ctx* c = &h->c;
    if (n_atoms > c->max_atoms) return DHP_E_CAPACITY;
    dhp_md* md = new (std::nothrow) dhp_md();
    if (!md) return DHP_E_NOMEM;
    Md* m = &md->m;
    memset((void*)m, 0, sizeof(Md));
    m->n_atoms = n_atoms; m->n_bonds = n_bonds;
    const size_t N = (size_t)n_atoms, NB = (size_t)(n_bonds > 0 ? n_bonds : 1);
    bool ok = cudaMalloc((void**)&m->inv_mass, sizeof(float) * N) == cudaSuccess && cudaMalloc((void**)&m->bonds, sizeof(int) * 2 * NB) == cudaSuccess &&
              cudaMalloc((void**)&m->bond_k, sizeof(float) * NB) == cudaSuccess && cudaMalloc((void**)&m->bond_r0, sizeof(float) * NB) == cudaSuccess &&
              cudaMalloc((void**)&m->f_slow, sizeof(float) * 3 * N) == cudaSuccess && cudaMalloc((void**)&m->f_fast, sizeof(float) * 3 * N) == cudaSuccess &&
              cudaMalloc((void**)&m->e, sizeof(double) * 3) == cudaSuccess;
    cudaStream_t st = c->stream;
    if (ok) ok = cudaMemcpyAsync(m->inv_mass, inv_mass, sizeof(float) * N, cudaMemcpyDefault, st) == cudaSuccess;
    if (ok && n_bonds > 0)
        ok = cudaMemcpyAsync(m->bonds, bonds, sizeof(int) * 2 * NB, cudaMemcpyDefault, st) == cudaSuccess &&
             cudaMemcpyAsync(m->bond_k, bond_k, sizeof(float) * NB, cudaMemcpyDefault, st) == cudaSuccess &&
             cudaMemcpyAsync(m->bond_r0, bond_r0, sizeof(float) * NB, cudaMemcpyDefault, st) == cudaSuccess;
    if (ok) ok = cudaMemsetAsync(m->e, 0, sizeof(double) * 3, st) == cudaSuccess && cudaMemsetAsync(m->f_fast, 0, sizeof(float) * 3 * N, st) == cudaSuccess &&
                 cudaStreamSynchronize(st) == cudaSuccess;
    if (!ok) {
        cudaGetLastError();
        for (void* p : {(void*)m->inv_mass, (void*)m->bonds, (void*)m->bond_k, (void*)m->bond_r0, (void*)m->f_slow, (void*)m->f_fast, (void*)m->e}) if (p) cudaFree(p);
        delete md;
        return DHP_E_NOMEM;
    }
    *out = md;
    return DHP_OK;
}

int dhp_md_destroy(dhp_ctx* h, dhp_md* md) {
    if (!h || !md) return DHP_E_BADARG;
    cudaStreamSynchronize(h->c.stream);
    Md* m = &md->m;
    for (void* p : {(void*)m->inv_mass, (void*)m->bonds, (void*)m->bond_k, (void*)m->bond_r0, (void*)m->f_slow, (void*)m->f_fast, (void*)m->e}) if (p) cudaFree(p);
    delete md;
    return DHP_OK;
}

int dhp_md_reset(dhp_ctx* h, dhp_md* md) {
    if (!h || !md) return DHP_E_BADARG;
    md->m.primed = false;
    return DHP_OK;
}

int dhp_md_run(dhp_ctx* h, dhp_md* md, float* pos, float* vel, const float* box, const int32_t* species,
               const dhp_weights* weights, int n_models, float dt, int n_inner, int n_steps, double* E_out) {
    if (!h || !md || !pos || !vel || !species || !weights || n_inner < 1 || n_steps < 0 || !(dt > 0.f)) return DHP_E_BADARG;
    Ctx* c = &h->c;
    Md* m = &md->m;
    const int64_t n = m->n_atoms;
    const int n3 = (int)(3 * n), nb = (n3 + 255) / 256;
    const float* ff = m->n_bonds > 0 ? m->f_fast : nullptr;
    if (m->n_bonds == 0) n_inner = 1;                     // nothing in the inner loop: plain velocity Verlet
    const float d = dt / (float)n_inner;
    int rc;
    if (!m->primed) {
        if ((rc = dhp_ani_energy_forces(h, pos, box, species, n, nullptr, 0, weights, n_models, m->e, m->f_slow)) != DHP_OK) return rc;
        if ((rc = fast_forces(c, m, pos, box)) != DHP_OK) return rc;
        m->primed = true;
    }
    for (int s = 0; s < n_steps; ++s) {
        for (int k = 0; k < n_inner; ++k) {
            // k = 0: the outer half kick rides along; k > 0: the closing half kick of inner step k-1 and the opening
            // one of step k use the same fast force, so they are one kick of d
            DHP_LAUNCH(c, k_md_kick_drift, nb, 256, 0, pos, vel, m->inv_mass, k == 0 ? m->f_slow : (const float*)nullptr, 0.5f * dt, ff,
                       k == 0 ? 0.5f * d : d, d, n3);
            if ((rc = fast_forces(c, m, pos, box)) != DHP_OK) return rc;
        }
        if ((rc = dhp_ani_energy_forces(h, pos, box, species, n, nullptr, 0, weights, n_models, m->e, m->f_slow)) != DHP_OK) return rc;
        DHP_LAUNCH(c, k_md_kick_drift, nb, 256, 0, pos, vel, m->inv_mass, m->f_slow, 0.5f * dt, ff, 0.5f * d, 0.f, n3);
    }
    if (E_out) {
        DHP_CUDA(c, cudaMemsetAsync(m->e + 2, 0, sizeof(double), c->stream));
        DHP_LAUNCH(c, k_md_kinetic, 2 * c->sm_count, 256, 0, vel, m->inv_mass, (int)n, m->e + 2);
        DHP_CUDA(c, cudaMemcpyAsync(E_out, m->e, sizeof(double) * 3, cudaMemcpyDeviceToDevice, c->stream));
    }
    DHP_CUDA(c, cudaGetLastError());
    return DHP_OK;
}

// ---- one outer step split at the slow-force evaluation, over the atoms [lo, hi) a rank owns (multi-GPU decomposition,
// PAPER.md L134 / L194): dhp_md_open = first half kick with the slow force + the whole inner loop (the
// rank's own bonds: both atoms of every bond of this md handle must lie in [lo, hi)), dhp_md_close = second half kick.
// Between the two the caller all-gathers the positions, evaluates its partial slow force (dhp_ani_energy_forces_partial)
// and reduce-scatters it (paper_2207_14276_b200/shard.py).  F_slow is dev fp32 [n_atoms][3]; only rows [lo, hi) are read.
int dhp_md_open(dhp_ctx* h, dhp_md* md, float* pos, float* vel, const float* box, const float* F_slow, float dt, int n_inner,
                int64_t lo, int64_t hi) {
    if (!h || !md || !pos || !vel || !F_slow || n_inner < 1 || !(dt > 0.f)) return DHP_E_BADARG;
    Ctx* c = &h->c;
    Md* m = &md->m;
    if (lo < 0 || hi < lo || hi > m->n_atoms) return DHP_E_BADARG;
    if (hi == lo) return DHP_OK;
    const int t0 = (int)(3 * lo), t1 = (int)(3 * hi), nb = (t1 - t0 + 255) / 256;
    const float* ff = m->n_bonds > 0 ? m->f_fast : nullptr;
    if (m->n_bonds == 0) n_inner = 1;
    const float d = dt / (float)n_inner;
    int rc;
    if (!m->primed) {                                    // fast force at the starting positions
        if ((rc = fast_forces(c, m, pos, box)) != DHP_OK) return rc;
        m->primed = true;
    }
    for (int k = 0; k < n_inner; ++k) {
        DHP_LAUNCH(c, k_md_kick_drift, nb, 256, 0, pos, vel, m->inv_mass, k == 0 ? F_slow : (const float*)nullptr, 0.5f * dt, ff,
                   k == 0 ? 0.5f * d : d, d, t1, t0);
        if ((rc = fast_forces(c, m, pos, box)) != DHP_OK) return rc;
    }
    m->open_dt = dt; m->open_n_inner = n_inner;           // the last fast half kick is dhp_md_close's: it needs the same d
    DHP_CUDA(c, cudaGetLastError());
    return DHP_OK;
}

int dhp_md_close(dhp_ctx* h, dhp_md* md, float* vel, const float* F_slow, float dt, int n_inner, int64_t lo, int64_t hi) {
    if (!h || !md || !vel || !F_slow || n_inner < 1 || !(dt > 0.f)) return DHP_E_BADARG;
    Ctx* c = &h->c;
    Md* m = &md->m;
    if (lo < 0 || hi < lo || hi > m->n_atoms) return DHP_E_BADARG;
    if (hi == lo) return DHP_OK;
    const int t0 = (int)(3 * lo), t1 = (int)(3 * hi), nb = (t1 - t0 + 255) / 256;
    const float* ff = m->n_bonds > 0 ? m->f_fast : nullptr;
    if (m->n_bonds == 0) n_inner = 1;
    // close finishes the step open began: another dt or n_inner would apply the pending fast half kick with the wrong length
    if (m->open_dt == 0.f || m->open_dt != dt || m->open_n_inner != n_inner) return DHP_E_BADARG;
    m->open_dt = 0.f;
    const float d = dt / (float)n_inner;
    DHP_LAUNCH(c, k_md_kick_drift, nb, 256, 0, (float*)nullptr, vel, m->inv_mass, F_slow, 0.5f * dt, ff, 0.5f * d, 0.f, t1, t0);
    DHP_CUDA(c, cudaGetLastError());
    return DHP_OK;
}


}  // extern "C"

// ---- kinetic energy for callers that may not allocate (include/dhp.h: dhp_kinetic_energy_static) ------------------------
// Same sum as k_md_kinetic, E_kin = sum_i 1/2 |v_i|^2 / inv_mass_i in fp64, but nothing here comes from cudaMalloc.
// k_md_kinetic adds into an accumulator that dhp_md_create allocated; this variant keeps its working memory - one partial
// sum per block and an arrival counter - in a fixed array that is part of the library image, so the entry point needs no
// context, no handle and no allocator.  The price is a size limit and a single shared copy per GPU (see the header).
namespace dhp {

constexpr int KIN_THREADS = 256;
constexpr int KIN_MAX_BLOCKS = DHP_KINETIC_STATIC_MAX_ATOMS / KIN_THREADS;   // one block per 256 atoms, one partial per block
constexpr int KIN_HEAD = 32;                                                 // doubles in front of the partials: 256 bytes for the counter
static_assert(DHP_KINETIC_STATIC_MAX_ATOMS % KIN_THREADS == 0, "whole blocks");

// [0] (as unsigned): number of blocks of the running call that have stored their partial; [KIN_HEAD + b]: partial sum of block b.
// 33 KB, resident on every GPU that has loaded libdhp.so for as long as the process lives.  On the host this name is only a
// handle for cudaGetSymbolAddress - it is NOT the device address and must never be handed to a kernel as it stands.
static __device__ __align__(256) double g_kin_scratch[KIN_HEAD + KIN_MAX_BLOCKS];

__global__ void __launch_bounds__(KIN_THREADS)
k_md_kinetic_static(const float* __restrict__ vel, const float* __restrict__ inv_mass, int n, double* __restrict__ scratch,
                    double* __restrict__ E_kin) {
    __shared__ double wsum[KIN_THREADS / 32];
    __shared__ bool last;
    const int tid = threadIdx.x, i = blockIdx.x * KIN_THREADS + tid;
    double e = 0.0;
    if (i < n) {
        const double vx = vel[3 * i], vy = vel[3 * i + 1], vz = vel[3 * i + 2];
        e = 0.5 * (vx * vx + vy * vy + vz * vz) / (double)inv_mass[i];
    }
    for (int o = 16; o; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
    if ((tid & 31) == 0) wsum[tid >> 5] = e;
    __syncthreads();
    if (tid == 0) {
        double b = 0.0;
        for (int w = 0; w < KIN_THREADS / 32; ++w) b += wsum[w];
        scratch[KIN_HEAD + blockIdx.x] = b;
        __threadfence();                                                     // the partial is visible before the arrival is counted
        last = atomicAdd((unsigned*)scratch, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    // the block that arrives last adds the partials in block order: the result does not depend on which block that was
    __threadfence();
    double t = 0.0;
    for (int b = tid; b < (int)gridDim.x; b += KIN_THREADS) t += __ldcg(&scratch[KIN_HEAD + b]);
    for (int o = 16; o; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    if ((tid & 31) == 0) wsum[tid >> 5] = t;
    __syncthreads();
    if (tid == 0) {
        double tot = 0.0;
        for (int w = 0; w < KIN_THREADS / 32; ++w) tot += wsum[w];
        *E_kin = tot;
        *(unsigned*)scratch = 0u;                                            // leave the counter as the next call expects it
    }
}

// Device address of g_kin_scratch per device ordinal, looked up once per device with that device current.
constexpr int KIN_MAX_DEVICES = 64;
static std::mutex g_kin_mu;
static double* g_kin_addr[KIN_MAX_DEVICES];

static cudaError_t kin_scratch_address(double** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const bool cached = dev >= 0 && dev < KIN_MAX_DEVICES;
    std::lock_guard<std::mutex> lock(g_kin_mu);
    if (cached && g_kin_addr[dev]) { *out = g_kin_addr[dev]; return cudaSuccess; }
    double* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_kin_scratch);                     // the address on the CURRENT device
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    if (cached) g_kin_addr[dev] = p;
    *out = p;
    return cudaSuccess;
}

}  // namespace dhp

extern "C" {

int dhp_kinetic_energy_static(const float* vel, const float* inv_mass, int64_t n_atoms, double* E_kin, void* cuda_stream) {
    if (!E_kin || n_atoms < 0 || (n_atoms > 0 && (!vel || !inv_mass))) return DHP_E_BADARG;
    if (n_atoms > DHP_KINETIC_STATIC_MAX_ATOMS) return DHP_E_CAPACITY;       // more blocks than the fixed array has partials for
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (n_atoms == 0) return cudaMemsetAsync(E_kin, 0, sizeof(double), st) == cudaSuccess ? DHP_OK : DHP_E_CUDA;
    double* scratch = nullptr;
    if (kin_scratch_address(&scratch) != cudaSuccess) { cudaGetLastError(); return DHP_E_CUDA; }
    // the array keeps whatever the previous call left: the counter has to read zero when the first block arrives, also after
    // a call that was cut short; the partials need no clearing, every block of this call overwrites its own before it is read
    if (cudaMemsetAsync(scratch, 0, sizeof(double) * KIN_HEAD, st) != cudaSuccess) { cudaGetLastError(); return DHP_E_CUDA; }
    const int blocks = (int)((n_atoms + KIN_THREADS - 1) / KIN_THREADS);
    k_md_kinetic_static<<<blocks, KIN_THREADS, 0, st>>>(vel, inv_mass, (int)n_atoms, scratch, E_kin);
    return cudaGetLastError() == cudaSuccess ? DHP_OK : DHP_E_CUDA;
}

}  // extern "C"
