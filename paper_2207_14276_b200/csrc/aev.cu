// a2 — AEV forward (Eqs. 3-5) and a5 — AEV backward (forces).
//
// One warp per central atom (sorted order, so the warps of a block share neighbours in L1/L2).
// Displacements are formed in fp64 from the fp32 inputs (exact difference, exact image shift) and
// rounded once to fp32; everything after that is fp32.  sin(theta) is |r_hat_ij x r_hat_ik|, never
// sqrt(1 - cos^2) (SURVEY.md §7 hard part 2).
//
// Forward, angular part, two phases per round of 32 triplets:
//   phase 1  lane <-> triplet (j,k): geometry, the 4 angular factors 2 u_z^zeta f_j f_k and the 8 radial
//            Gaussians (12 values, the minimum number of MUFU ops), staged in shared memory;
//   phase 2  lane <-> feature (a,z): for each staged triplet, acc[pair(s_j,s_k)][a][z] += A_z B_a into a
//            warp-private shared row (lane-private address: no atomics, no conflicts).
// Backward: "distance rounds" d = 1..n/2 with j = lane, k = (j + d) mod n, so that within a round all j
// are distinct and all k are distinct and the per-neighbour force accumulators in shared memory are
// updated without atomics; one global atomic triple per neighbour at the end.
#include <algorithm>

#include "dhp_internal.cuh"

namespace dhp {

constexpr int AEV_WARPS = 4;
constexpr int GP = 36;   // pitch of one 32-float angular block of the staged gradient row (bank spread, 16 B aligned)

__device__ __forceinline__ float fast_exp2(float x) { return exp2f(x); }     // ex2.approx under -use_fast_math
__device__ __forceinline__ float fast_log2(float x) { return __log2f(x); }

struct NbrGeom {
    float ux, uy, uz, R;
    int sp;
};

// displacement r_j - r_i with the minimum image, fp64 -> fp32 (one rounding per component)
__device__ __forceinline__ NbrGeom neighbour_geom(const float4& pi, const float4& pj, const Grid& g) {
    double d[3] = {(double)pj.x - (double)pi.x, (double)pj.y - (double)pi.y, (double)pj.z - (double)pi.z};
    if (g.periodic) {
#pragma unroll
        for (int c = 0; c < 3; ++c) d[c] -= g.L[c] * rint(d[c] / g.L[c]);
    }
    float x = (float)d[0], y = (float)d[1], z = (float)d[2];
    float r2 = x * x + y * y + z * z;
    float inv = rsqrtf(r2);
    inv = inv * (1.5f - 0.5f * r2 * inv * inv);          // one Newton step: full fp32 accuracy
    NbrGeom o;
    o.R = r2 * inv;
    o.ux = x * inv; o.uy = y * inv; o.uz = z * inv;
    o.sp = __float_as_int(pj.w);
    return o;
}

// Eq. 3: f_c(R) = 1/2 cos(pi R / Rc) + 1/2 (R <= Rc is guaranteed by the pair list)
__device__ __forceinline__ float fcut(float R, float inv_rc) { return 0.5f * cospif(R * inv_rc) + 0.5f; }
__device__ __forceinline__ float dfcut(float R, float inv_rc, float pi_over_rc) { return -0.5f * pi_over_rc * sinpif(R * inv_rc); }

struct WarpSmemFwd {
    float rad[2][AEV_RAD];
    float ang[AEV_ANG];
    float ux[MAX_ANG], uy[MAX_ANG], uz[MAX_ANG], R[MAX_ANG], fc[MAX_ANG];
    int sp[MAX_ANG];
    float4 tA[32];
    float4 tB[32][2];
    int tp[32];
};

__global__ void __launch_bounds__(AEV_WARPS * 32)
k_aev_fwd(const float4* __restrict__ spos, const int* __restrict__ row_ptr, const int* __restrict__ col,
          const int* __restrict__ n_ang, const int* __restrict__ rowmap, const Grid* __restrict__ gp,
          const __grid_constant__ AevConst K, int n, float* __restrict__ aev, int* __restrict__ status) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ Grid g;
    if (threadIdx.x == 0) g = *gp;
    __syncthreads();
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int i = blockIdx.x * AEV_WARPS + w;
    if (i >= n) return;
    WarpSmemFwd& S = reinterpret_cast<WarpSmemFwd*>(smem_raw)[w];

    for (int c = lane; c < 2 * AEV_RAD; c += 32) (&S.rad[0][0])[c] = 0.f;
    for (int c = lane; c < AEV_ANG; c += 32) S.ang[c] = 0.f;
    __syncwarp();

    const float4 pi = spos[i];
    const int rb = row_ptr[i], re = row_ptr[i + 1];
    int na = n_ang[i];
    if (na > MAX_ANG) { if (lane == 0) atomicExch(status, DHP_E_CAPACITY); na = MAX_ANG; }
    const float inv_rcr = 1.0f / K.rcr, inv_rca = 1.0f / K.rca;
    const int m = lane & 15, half = lane >> 4;
    const float shf = K.shf_r[m];

    // ---- radial (Eq. 4) + staging of the angular neighbours --------------------------------------
    for (int base = rb; base < re; base += 32) {
        const int idx = base + lane;
        NbrGeom q; q.R = 1.f; q.sp = 0; q.ux = q.uy = q.uz = 0.f;
        float fc = 0.f;
        if (idx < re) {
            q = neighbour_geom(pi, spos[col[idx]], g);
            fc = fcut(q.R, inv_rcr);
            const int a = idx - rb;
            if (a < na) {
                S.ux[a] = q.ux; S.uy[a] = q.uy; S.uz[a] = q.uz; S.R[a] = q.R; S.sp[a] = q.sp;
                S.fc[a] = fcut(q.R, inv_rca);
            }
        }
        const int cnt = min(32, re - base);
        for (int t = 0; t < cnt; t += 2) {
            const int src = t + half;
            float Rq = __shfl_sync(0xffffffffu, q.R, src & 31);
            float fq = __shfl_sync(0xffffffffu, fc, src & 31);
            int sq = __shfl_sync(0xffffffffu, q.sp, src & 31);
            if (src < cnt) {
                float dr = Rq - shf;
                S.rad[half][NR * sq + m] += fast_exp2(-K.eta_r_l2e * dr * dr) * fq;
            }
        }
    }
    __syncwarp();

    // ---- angular (Eq. 5) ---------------------------------------------------------------------------
    const int npairs = na * (na - 1) / 2;
    const float inv_na = na > 0 ? 1.0f / (float)na : 0.f;
    const int za = lane & 3, aa = lane >> 2;
    for (int T0 = 0; T0 < npairs; T0 += 32) {
        const int T = T0 + lane;
        if (T < npairs) {
            int d = (int)(((float)T + 0.5f) * inv_na);
            int j = T - d * na;
            if (j < 0) { --d; j += na; } else if (j >= na) { ++d; j -= na; }
            int k = j + d + 1;
            if (k >= na) k -= na;
            float ujx = S.ux[j], ujy = S.uy[j], ujz = S.uz[j];
            float ukx = S.ux[k], uky = S.uy[k], ukz = S.uz[k];
            float c = ujx * ukx + ujy * uky + ujz * ukz;
            float cx = ujy * ukz - ujz * uky, cy = ujz * ukx - ujx * ukz, cz = ujx * uky - ujy * ukx;
            float s = sqrtf(cx * cx + cy * cy + cz * cz);
            float f2 = 2.0f * S.fc[j] * S.fc[k];
            float Rm = 0.5f * (S.R[j] + S.R[k]);
            float A[NZ];
#pragma unroll
            for (int z = 0; z < NZ; ++z) {
                float u = fmaxf(0.5f * (1.0f + c * K.cos_z[z] + s * K.sin_z[z]), 0.f);
                A[z] = f2 * fast_exp2(K.zeta * fast_log2(u));        // 2 ((1+cos(theta-theta_z))/2)^zeta f_j f_k
            }
            float B[NA];
#pragma unroll
            for (int a = 0; a < NA; ++a) {
                float mm = Rm - K.shf_a[a];
                B[a] = fast_exp2(-K.eta_a_l2e * mm * mm);
            }
            S.tA[lane] = make_float4(A[0], A[1], A[2], A[3]);
            S.tB[lane][0] = make_float4(B[0], B[1], B[2], B[3]);
            S.tB[lane][1] = make_float4(B[4], B[5], B[6], B[7]);
            S.tp[lane] = ipair(S.sp[j], S.sp[k]);
        }
        __syncwarp();
        const int cnt = min(32, npairs - T0);
        const float* tA = reinterpret_cast<const float*>(S.tA);
        const float* tB = reinterpret_cast<const float*>(S.tB);
        for (int t = 0; t < cnt; ++t) {
            float v = tA[4 * t + za] * tB[8 * t + aa];
            S.ang[32 * S.tp[t] + lane] += v;                        // lane == 4*aa + za: layout [a][z]
        }
        __syncwarp();
    }

    // ---- write the row (species-grouped row order) -------------------------------------------------
    float* out = aev + (size_t)rowmap[i] * AEV_LD;
    // internal column order (dhp_internal.cuh): angular blocks by ipair(), radial blocks by species priority, zeros
    for (int c = lane; c < AEV_ANG; c += 32) out[c] = S.ang[c];
    for (int c = lane; c < AEV_RAD; c += 32) out[rad_col(c >> 4) + (c & 15)] = S.rad[0][c] + S.rad[1][c];
    if (lane < AEV_LD - AEV_DIM) out[AEV_DIM + lane] = 0.f;
}

// -------------------------------------------------------------------------------------------------
// backward
// -------------------------------------------------------------------------------------------------
struct WarpSmemBwd {
    float grad_rad[AEV_RAD];
    float grad_ang[NPAIR * GP];
    float ux[MAX_ANG], uy[MAX_ANG], uz[MAX_ANG], R[MAX_ANG], fc[MAX_ANG], dfc[MAX_ANG];
    float fx[MAX_ANG], fy[MAX_ANG], fz[MAX_ANG];
    int sp[MAX_ANG];
};

__global__ void __launch_bounds__(AEV_WARPS * 32)
k_aev_bwd(const float4* __restrict__ spos, const int* __restrict__ row_ptr, const int* __restrict__ col,
          const int* __restrict__ n_ang, const int* __restrict__ rowmap, const Grid* __restrict__ gp,
          const __grid_constant__ AevConst K, int n, const float* __restrict__ grad, float* __restrict__ fsorted) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ Grid g;
    if (threadIdx.x == 0) g = *gp;
    __syncthreads();
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int i = blockIdx.x * AEV_WARPS + w;
    if (i >= n) return;
    WarpSmemBwd& S = reinterpret_cast<WarpSmemBwd*>(smem_raw)[w];

    const float* grow = grad + (size_t)rowmap[i] * AEV_LD;
    for (int c = lane; c < AEV_RAD; c += 32) S.grad_rad[c] = grow[rad_col(c >> 4) + (c & 15)];
    for (int c = lane; c < AEV_ANG; c += 32) S.grad_ang[(c >> 5) * GP + (c & 31)] = grow[c];

    const float4 pi = spos[i];
    const int rb = row_ptr[i], re = row_ptr[i + 1];
    const int na = min(n_ang[i], MAX_ANG);
    const float inv_rcr = 1.0f / K.rcr, inv_rca = 1.0f / K.rca;

    // stage the angular neighbours (the prefix of the row)
    for (int a = lane; a < na; a += 32) {
        NbrGeom q = neighbour_geom(pi, spos[col[rb + a]], g);
        S.ux[a] = q.ux; S.uy[a] = q.uy; S.uz[a] = q.uz; S.R[a] = q.R; S.sp[a] = q.sp;
        S.fc[a] = fcut(q.R, inv_rca);
        S.dfc[a] = dfcut(q.R, inv_rca, K.pi_over_rca);
        S.fx[a] = 0.f; S.fy[a] = 0.f; S.fz[a] = 0.f;
    }
    __syncwarp();

    float fix = 0.f, fiy = 0.f, fiz = 0.f;     // force on the centre, summed over this lane's terms

    // ---- angular: rounds over the index distance d ---------------------------------------------------
    for (int d = 1; 2 * d <= na; ++d) {
        const int jmax = (2 * d == na) ? na / 2 : na;     // even n: the last round holds each pair once
        for (int jb = 0; jb < jmax; jb += 32) {
            const int j = jb + lane;
            const bool act = j < jmax;
            int k = 0;
            float gjx = 0.f, gjy = 0.f, gjz = 0.f, gkx = 0.f, gky = 0.f, gkz = 0.f;
            if (act) {
                k = j + d; if (k >= na) k -= na;
                const float ujx = S.ux[j], ujy = S.uy[j], ujz = S.uz[j], Rj = S.R[j];
                const float ukx = S.ux[k], uky = S.uy[k], ukz = S.uz[k], Rk = S.R[k];
                const float c = ujx * ukx + ujy * uky + ujz * ukz;
                const float cx = ujy * ukz - ujz * uky, cy = ujz * ukx - ujx * ukz, cz = ujx * uky - ujy * ukx;
                const float s = sqrtf(cx * cx + cy * cy + cz * cz);
                const float fj = S.fc[j], fk = S.fc[k], dfj = S.dfc[j], dfk = S.dfc[k];
                const float Rm = 0.5f * (Rj + Rk);
                const float* gb = &S.grad_ang[GP * ipair(S.sp[j], S.sp[k])];
                float Az[NZ], dAz[NZ];
#pragma unroll
                for (int z = 0; z < NZ; ++z) {
                    float u = fmaxf(0.5f * (1.0f + c * K.cos_z[z] + s * K.sin_z[z]), 0.f);
                    float wz = fast_exp2((K.zeta - 1.0f) * fast_log2(u));      // u^(zeta-1)
                    Az[z] = 2.0f * u * wz;                                      // A = 2 u^zeta
                    dAz[z] = -K.zeta * wz * (s * K.cos_z[z] - c * K.sin_z[z]);  // dA/dtheta
                }
                float S0 = 0.f, Sm = 0.f, St = 0.f;
#pragma unroll
                for (int a = 0; a < NA; ++a) {
                    const float4 g4 = *reinterpret_cast<const float4*>(gb + 4 * a);
                    float mm = Rm - K.shf_a[a];
                    float B = fast_exp2(-K.eta_a_l2e * mm * mm);
                    float dB = -K.eta_a * mm * B;                               // dB/dR_ij = dB/dR_ik
                    float ua = g4.x * Az[0] + g4.y * Az[1] + g4.z * Az[2] + g4.w * Az[3];
                    float va = g4.x * dAz[0] + g4.y * dAz[1] + g4.z * dAz[2] + g4.w * dAz[3];
                    S0 += B * ua; Sm += dB * ua; St += B * va;
                }
                const float dth = St * fj * fk;                                 // sum g dT/dtheta
                const float dRj = (Sm * fj + S0 * dfj) * fk;                    // sum g dT/dR_ij
                const float dRk = (Sm * fk + S0 * dfk) * fj;
                const float inv_s = s > 1e-20f ? 1.0f / s : 0.f;                // collinear: e = 0 (Q7)
                const float tj = -dth * inv_s / Rj, tk = -dth * inv_s / Rk;     // d theta/d r_j = -e_j / R_ij
                gjx = tj * (ukx - c * ujx) + dRj * ujx; gjy = tj * (uky - c * ujy) + dRj * ujy; gjz = tj * (ukz - c * ujz) + dRj * ujz;
                gkx = tk * (ujx - c * ukx) + dRk * ukx; gky = tk * (ujy - c * uky) + dRk * uky; gkz = tk * (ujz - c * ukz) + dRk * ukz;
                fix += gjx + gkx; fiy += gjy + gky; fiz += gjz + gkz;
                S.fx[j] -= gjx; S.fy[j] -= gjy; S.fz[j] -= gjz;                 // all j distinct in this step
            }
            __syncwarp();
            if (act) { S.fx[k] -= gkx; S.fy[k] -= gky; S.fz[k] -= gkz; }       // all k distinct in this step
            __syncwarp();
        }
    }

    // ---- radial + scatter ----------------------------------------------------------------------------
    for (int base = rb; base < re; base += 32) {
        const int idx = base + lane;
        if (idx < re) {
            const int j = col[idx];
            NbrGeom q = neighbour_geom(pi, spos[j], g);
            const float fc = fcut(q.R, inv_rcr), dfc = dfcut(q.R, inv_rcr, K.pi_over_rcr);
            const float* gr = &S.grad_rad[NR * q.sp];
            float coef = 0.f;
#pragma unroll
            for (int mI = 0; mI < NR; ++mI) {
                float dr = q.R - K.shf_r[mI];
                float t = fast_exp2(-K.eta_r_l2e * dr * dr);
                coef += gr[mI] * t * (-2.0f * K.eta_r * dr * fc + dfc);
            }
            float vx = coef * q.ux, vy = coef * q.uy, vz = coef * q.uz;
            fix += vx; fiy += vy; fiz += vz;
            float fjx = -vx, fjy = -vy, fjz = -vz;
            const int a = idx - rb;
            if (a < na) { fjx += S.fx[a]; fjy += S.fy[a]; fjz += S.fz[a]; }
            atomicAdd(&fsorted[3 * j + 0], fjx);
            atomicAdd(&fsorted[3 * j + 1], fjy);
            atomicAdd(&fsorted[3 * j + 2], fjz);
        }
    }
    for (int o = 16; o; o >>= 1) {
        fix += __shfl_xor_sync(0xffffffffu, fix, o);
        fiy += __shfl_xor_sync(0xffffffffu, fiy, o);
        fiz += __shfl_xor_sync(0xffffffffu, fiz, o);
    }
    if (lane == 0) {
        atomicAdd(&fsorted[3 * i + 0], fix);
        atomicAdd(&fsorted[3 * i + 1], fiy);
        atomicAdd(&fsorted[3 * i + 2], fiz);
    }
}

__global__ void k_unsort_forces(const float* __restrict__ fsorted, const int* __restrict__ perm, int n, float* __restrict__ F) {
    int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= n) return;
    int i = perm[a];
    F[3 * i + 0] = fsorted[3 * a + 0];
    F[3 * i + 1] = fsorted[3 * a + 1];
    F[3 * i + 2] = fsorted[3 * a + 2];
}

// E (per molecule, or one total): fp64 sum of the per-row atomic energies
__global__ void k_energy_reduce(const float* __restrict__ e_atom, const int* __restrict__ row_slot,
                                const int* __restrict__ smol, const int* __restrict__ sp_start, int per_mol,
                                double* __restrict__ E) {
    __shared__ double part[32];
    const int nrows = sp_start[NSP];
    double acc = 0.0;
    for (int r = blockIdx.x * blockDim.x + threadIdx.x; r < nrows; r += gridDim.x * blockDim.x) {
        int slot = row_slot[r];
        if (slot < 0) continue;
        double e = (double)e_atom[r];
        if (per_mol) atomicAdd(&E[smol[slot]], e);
        else acc += e;
    }
    if (per_mol) return;
    for (int o = 16; o; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x < 32) {
        double v = threadIdx.x < (blockDim.x >> 5) ? part[threadIdx.x] : 0.0;
        for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (threadIdx.x == 0) atomicAdd(E, v);
    }
}

// -------------------------------------------------------------------------------------------------
int aev_forward(Ctx* ctx) {
    const int n = (int)ctx->n_atoms;
    if (n == 0) return DHP_OK;
    static bool attr_set = false;
    const size_t smem = sizeof(WarpSmemFwd) * AEV_WARPS;
    if (!attr_set) {
        DHP_CUDA(ctx, cudaFuncSetAttribute(k_aev_fwd, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_set = true;
    }
    DHP_LAUNCH(ctx, k_aev_fwd, (n + AEV_WARPS - 1) / AEV_WARPS, AEV_WARPS * 32, smem, ctx->spos, ctx->row_ptr, ctx->col,
               ctx->n_ang, ctx->rowmap, ctx->grid, ctx->aevc, n, ctx->aev, ctx->status);
    DHP_CUDA(ctx, cudaGetLastError());
    return DHP_OK;
}

int aev_backward(Ctx* ctx, float* F_out) {
    const int n = (int)ctx->n_atoms;
    if (n == 0) return DHP_OK;
    static bool attr_set = false;
    const size_t smem = sizeof(WarpSmemBwd) * AEV_WARPS;
    if (!attr_set) {
        DHP_CUDA(ctx, cudaFuncSetAttribute(k_aev_bwd, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_set = true;
    }
    DHP_CUDA(ctx, cudaMemsetAsync(ctx->fsorted, 0, sizeof(float) * 3 * n, ctx->stream));
    DHP_LAUNCH(ctx, k_aev_bwd, (n + AEV_WARPS - 1) / AEV_WARPS, AEV_WARPS * 32, smem, ctx->spos, ctx->row_ptr, ctx->col,
               ctx->n_ang, ctx->rowmap, ctx->grid, ctx->aevc, n, ctx->grad, ctx->fsorted);
    DHP_LAUNCH(ctx, k_unsort_forces, (n + 255) / 256, 256, 0, ctx->fsorted, ctx->perm, n, F_out);
    DHP_CUDA(ctx, cudaGetLastError());
    return DHP_OK;
}

int energy_reduce(Ctx* ctx, double* E_out) {
    const int per_mol = ctx->n_mol > 0 ? 1 : 0;
    const int64_t ne = per_mol ? ctx->n_mol : 1;
    DHP_CUDA(ctx, cudaMemsetAsync(E_out, 0, sizeof(double) * ne, ctx->stream));
    if (ctx->n_atoms == 0) return DHP_OK;
    int blocks = (int)std::min<int64_t>((ctx->n_atoms + 255) / 256 + NSP, 2 * ctx->sm_count);
    DHP_LAUNCH(ctx, k_energy_reduce, blocks, 256, 0, ctx->e_atom, ctx->row_slot, ctx->smol, ctx->sp_start, per_mol, E_out);
    DHP_CUDA(ctx, cudaGetLastError());
    return DHP_OK;
}

}  // namespace dhp
