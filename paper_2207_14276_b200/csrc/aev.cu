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
#include <cstdlib>

#include "dhp_internal.cuh"

namespace dhp {


// single-instruction approximations (2^-22 relative error; inputs here are never denormal where it matters)
__device__ __forceinline__ float fast_exp2(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float fast_log2(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float fast_sqrt(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float fast_rcp(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// Blackwell's packed fp32 pipe: one FFMA2 does two fp32 FMAs (the AEV kernels are bound by instruction issue, not by a pipe).
// A pair is a 64-bit register; when both halves of an operand are the same value ptxas uses the scalar-broadcast form.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float a, float b) { f32x2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void unpack2(f32x2 v, float& a, float& b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) { f32x2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) { f32x2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }

struct NbrGeom {
    float ux, uy, uz, R;
    int sp;
};

// displacement r_j - r_i with the minimum image, fp64 -> fp32 (one rounding per component)
__device__ __forceinline__ NbrGeom neighbour_geom(const float4& pi, const float4& pj, const Grid& g) {
    double d[3] = {(double)pj.x - (double)pi.x, (double)pj.y - (double)pi.y, (double)pj.z - (double)pi.z};
    if (g.periodic) {
#pragma unroll
        for (int c = 0; c < 3; ++c) d[c] -= g.L[c] * rint(d[c] * g.inv_L[c]);   // listed pairs are far from the half-box tie
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

// ---- forward ---------------------------------------------------------------------------------------
// Row i of the pair list is ordered [angular, species 0..6][radial-only, species 0..6] (nlist.cu), seg_cnt holds
// the 14 run lengths.  The kernel uses that order twice:
//   radial   lane = (shift m, parity h): a register sum over the two runs of each neighbour species;
//   angular  triplets are enumerated species pair by species pair (internal pair index p = angular block p of
//            the row), each pair padded to a multiple of 4 slots.  A round of 32 slots:
//              phase 1  lane <-> slot: geometry, 4 angular factors, 8 radial Gaussians -> staged [factor][slot];
//              phase 2  lane <-> feature (a,z): sum over the slots of each pair present in the round with
//                       16-byte broadcast reads (2 per 4 triplets), the sum carried in a register until the
//                       pair ends, then stored once to the row buffer (no read-modify-write, no atomics).
// Output: PLANES = false, full fp32 rows (SIMT MLP path); PLANES = true, the two-term fp16 split of the
// feature blocks that are active for the row's tile (what G1 reads), written straight into the tensor path's planes.
#ifndef AEV_ABL
#define AEV_ABL 0      // timing experiments only (wrong results): 1 = no radial loop, 2 = no phase-2 accumulation, 4 = no MUFU in the angular factors;
                       // backward: 16 = no radial derivative, 32 = no contraction with the dE/dG block, 64 = no gather, 128 = no angular rounds
#endif
#ifndef FWD_W
#define FWD_W 8
#endif
constexpr int AEV_WARPS = FWD_W;
constexpr int MAX_RAD = DHP_MAX_RAD;    // radial neighbours staged per centre (= the pair list's per-row capacity)

// internal pair p = hi (hi + 1) / 2 + lo over priority positions -> species(lo) | species(hi) << 4 (prio_sp(), dhp_internal.cuh);
// a static initialiser, so every device of the process has it without a per-device upload
#define DHP_PAIR_SP_TABLE {0, 48, 51, 16, 19, 17, 32, 35, 33, 34, 64, 67, 65, 66, 68, 80, 83, 81, 82, 84, 85, 96, 99, 97, 98, 100, 101, 102}
__constant__ unsigned char c_pair_sp[NPAIR] = DHP_PAIR_SP_TABLE;
static const unsigned char h_pair_sp[NPAIR] = DHP_PAIR_SP_TABLE;

constexpr int TP = 36;          // pitch of the staged factor rows: 16-byte aligned, rows 4 banks apart (conflict-free float4 reads)

struct __align__(16) WarpSmemFwd {
    float4 nb[MAX_ANG];          // ux, uy, uz, R of the angular neighbours
    float fca[MAX_ANG];          // f_c(R; Rca)
    union {                      // the radial part is finished before the first angular round is staged: same bytes
        float2 rr[MAX_RAD];      // all neighbours: R, f_c(R; Rcr)
        float st[12][TP];        // staged factor rows of one round: n_z angular rows, then n_a radial rows (8 + 4 or 4 + 8)
    };
    int4 tab[NPAIR + 1];         // non-empty species pairs in slot order: first slot, j0 | k0 << 8 | nk << 16 | same << 24,
                                 // triplets, angular block; terminated by {total slots, ...}
};

// one feature value of this lane -> the row, either fp32 or as the two-term fp16 split in the hi / lo planes
// Planes (tiled operand layout, aev_tiled_off()): `row_hi` points at (row, column 0) of the hi plane and `lane_off` is the lane's
// fixed part of the offset, so that a 32-column angular block blk costs one shift (its 64-column block and 8-column group
// fold into blk * 4096 halves) and a 16-column radial slot q one more (14 * 8192 + q * 2048).  AEV entries are sums of at
// most MAX_ANG^2 / 2 terms of at most 2: far inside the fp16 range, no clamp.
template <bool PLANES>
__device__ __forceinline__ void put_value(float v, float* __restrict__ row_f32, __half* __restrict__ row_hi, size_t plane_stride,
                                          int colidx, int tiled) {
    if (!PLANES) { row_f32[colidx] = v; return; }
    const __half hi = __float2half_rn(v);
    row_hi[tiled] = hi;
    row_hi[plane_stride + tiled] = __float2half_rn(v - __half2float(hi));
}
// angular block blk, column 32 blk + lane; lane_off = (lane >> 3) * 1024 + (lane & 7)
#define PUT_ANG(v, blk) put_value<PLANES>(v, row_f32, row_hi, plane_stride, 32 * (blk) + lane, ((blk) << 12) + lane_off)
// radial slot q (priority order), column AEV_ANG + 16 q + lane for lane < 16
#define PUT_RAD(v, q) put_value<PLANES>(v, row_f32, row_hi, plane_stride, AEV_ANG + 16 * (q) + lane, 14 * (ROW_TILE * KBLK) + ((q) << 11) + lane_off)

// SPLIT (small systems, n <= SMALL_N): one block of AEV_WARPS warps per atom, as in the backward kernel - warp 0 stages the neighbours
// and does the radial part, the angular rounds are dealt out to the warps (one warp per atom is latency-bound: ~3 k dependent
// instructions whatever the system size); each warp sums its rounds' pair blocks into a private shared row, the rows are added
// and written at the end.
template <bool PLANES, int NAg, int NZg, bool SPLIT>     // NAg x NZg: the angular grid of Eq. 5, 8 x 4 (ANI-2x shape) or 4 x 8 (ANI-1x shape)
__global__ void __launch_bounds__(AEV_WARPS * 32, SPLIT ? 1 : 40 / AEV_WARPS)
k_aev_fwd(const float4* __restrict__ spos, const int* __restrict__ row_ptr, const int* __restrict__ col,
          const unsigned short* __restrict__ seg_cnt, const int* __restrict__ rowmap, const unsigned* __restrict__ tile_mask,
          const Grid* __restrict__ gp, const __grid_constant__ AevConst K, int n, float* __restrict__ aev,
          __half* __restrict__ planes, size_t plane_stride, int* __restrict__ status, const int* __restrict__ row_slot) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ Grid g;
    if (threadIdx.x == 0) g = *gp;
    __syncthreads();
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    // full evaluation: warp <-> atom in sorted (cell) order, so that the warps of a block share neighbours; partial
    // evaluation (row_slot != null, n = an upper bound of the rows): warp <-> row, so that no warp is spent on the atoms
    // that are not central in this call
    int i = SPLIT ? (int)blockIdx.x : blockIdx.x * AEV_WARPS + w;
    if (i >= n) return;
    if (row_slot) { i = row_slot[i]; if (i < 0) return; }
    WarpSmemFwd& S = reinterpret_cast<WarpSmemFwd*>(smem_raw)[SPLIT ? 0 : w];       // geometry and pair table of the atom
    WarpSmemFwd& Sw = reinterpret_cast<WarpSmemFwd*>(smem_raw)[w];                   // this warp's staging rows
    float* part = reinterpret_cast<float*>(smem_raw + sizeof(WarpSmemFwd) * AEV_WARPS) + (size_t)w * (NPAIR * 32);   // SPLIT: this warp's pair-block sums
    const int sw = SPLIT ? w : 0;
    constexpr int NWARP = SPLIT ? AEV_WARPS : 1;
    const unsigned FULL = 0xffffffffu;
    const unsigned lt = (1u << lane) - 1u;

    // run lengths of the row: lane k < 7 angular species k, 8 <= k < 15 radial-only species k - 8
    int cnt = (lane < 16 && lane != 7 && lane != 15) ? (int)seg_cnt[(size_t)i * 16 + lane] : 0;
    int start = cnt;                                   // exclusive prefix over lanes = first slot of the run
#pragma unroll
    for (int o = 1; o < 16; o <<= 1) {
        int y = __shfl_up_sync(FULL, start, o);
        if (lane >= o) start += y;
    }
    start -= cnt;
    const int na = __shfl_sync(FULL, start, 8);        // angular neighbours = first slot of the radial-only class
    const int ntot = __shfl_sync(FULL, start, 15);
    if (na > MAX_ANG || ntot > MAX_RAD) {              // capacity: report it and produce a zero row
        if (lane == 0) atomicExch(status, DHP_E_CAPACITY);
        cnt = 0;
    }
    const int nst = (na > MAX_ANG || ntot > MAX_RAD) ? 0 : ntot;
    const int rb = row_ptr[i];
    const float4 pi = spos[i];
    const float inv_rcr = 1.0f / K.rcr, inv_rca = 1.0f / K.rca;
    const int row = rowmap[i];
    if (row < 0) return;                               // not a central atom of this call (partial evaluation)
    float* row_f32 = aev + (size_t)row * AEV_LD;
    __half* row_hi = planes + aev_tiled_off(row, 0);
    const int lane_off = (lane >> 3) * (ROW_TILE * 8) + (lane & 7);

    if (SPLIT) {
#pragma unroll
        for (int p = 0; p < NPAIR; ++p) part[p * 32 + lane] = 0.f;
    }
    // ---- stage all neighbours -------------------------------------------------------------------------
    for (int a = lane; a < (sw == 0 ? nst : 0); a += 32) {
        const NbrGeom q = neighbour_geom(pi, spos[col[rb + a]], g);
        S.rr[a] = make_float2(q.R, fcut(q.R, inv_rcr));
        if (a < na) {
            S.nb[a] = make_float4(q.ux, q.uy, q.uz, q.R);
            S.fca[a] = fcut(q.R, inv_rca);
        }
    }

    // ---- table of the non-empty species pairs (lane p < 28: internal pair p = angular block p) -------------
    int T_pad;
    unsigned nz_pairs;                                   // internal pairs with at least one triplet
    {
        int psa = 0, psb = 0, pcount = 0;
        if (lane < NPAIR) { const int e = c_pair_sp[lane]; psa = e & 15; psb = e >> 4; }
        const int ca = __shfl_sync(FULL, cnt, psa), cb = __shfl_sync(FULL, cnt, psb);
        const int ja0 = __shfl_sync(FULL, start, psa), kb0 = __shfl_sync(FULL, start, psb);
        if (lane < NPAIR) pcount = (psa == psb) ? ca * (ca - 1) / 2 : ca * cb;
        const int padded = (pcount + 3) & ~3;          // each pair padded to a multiple of 4 slots
        int pstart = padded;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int y = __shfl_up_sync(FULL, pstart, o);
            if (lane >= o) pstart += y;
        }
        T_pad = __shfl_sync(FULL, pstart, 31);
        pstart -= padded;
        const unsigned nz = __ballot_sync(FULL, pcount > 0);
        nz_pairs = nz;
        if (pcount > 0 && sw == 0) S.tab[__popc(nz & lt)] = make_int4(pstart, ja0 | (kb0 << 8) | (cb << 16) | ((psa == psb) << 24), pcount, lane);
        if (lane == 0 && sw == 0) S.tab[__popc(nz)] = make_int4(T_pad, 0, 0, 0);
    }
    __syncwarp();

    // ---- radial (Eq. 4): lane = (shift pair m2, neighbour phase h); the two Gaussians of a lane as one packed fp32 pair,
    //      one register sum per neighbour species; the 16 sums of a species leave as 8 packed stores per plane -------------
    {
        const int m2 = lane & 7, h = lane >> 3;
        const f32x2 nshf = pack2(-K.shf_r[2 * m2], -K.shf_r[2 * m2 + 1]);
        const f32x2 neta = pack2(-K.eta_r_l2e, -K.eta_r_l2e);
        for (int s = 0; s < (sw == 0 ? NSP : 0); ++s) {
            const int ca = __shfl_sync(FULL, cnt, s), sa = __shfl_sync(FULL, start, s);
            const int cr = __shfl_sync(FULL, cnt, 8 + s), sr = __shfl_sync(FULL, start, 8 + s) - ca;
            if (ca + cr == 0) continue;
            f32x2 acc = pack2(0.f, 0.f);
#pragma unroll 2
            for (int x = h; x < ((AEV_ABL & 1) ? 0 : ca + cr); x += 4) {
                const float2 q = S.rr[x < ca ? sa + x : sr + x];
                const f32x2 dr = add2(pack2(q.x, q.x), nshf);
                float a0, a1;
                unpack2(mul2(mul2(dr, neta), dr), a0, a1);
                acc = fma2(pack2(fast_exp2(a0), fast_exp2(a1)), pack2(q.y, q.y), acc);
            }
            float v0, v1;
            unpack2(acc, v0, v1);
            v0 += __shfl_xor_sync(FULL, v0, 8);  v1 += __shfl_xor_sync(FULL, v1, 8);
            v0 += __shfl_xor_sync(FULL, v0, 16); v1 += __shfl_xor_sync(FULL, v1, 16);
            if (lane < 8) {
                const int q = (rad_col(s) - AEV_ANG) >> 4;                 // radial slot (priority order), columns AEV_ANG + 16 q + 2 m2, + 1
                if (!PLANES) {
                    *reinterpret_cast<float2*>(row_f32 + AEV_ANG + 16 * q + 2 * m2) = make_float2(v0, v1);
                } else {
                    const int o = 14 * (ROW_TILE * KBLK) + (q << 11) + (m2 >> 2) * (ROW_TILE * 8) + 2 * (m2 & 3);
                    const __half2 hi = __floats2half2_rn(v0, v1);
                    const float2 hf = __half22float2(hi);
                    *reinterpret_cast<__half2*>(row_hi + o) = hi;
                    *reinterpret_cast<__half2*>(row_hi + plane_stride + o) = __floats2half2_rn(v0 - hf.x, v1 - hf.y);
                }
            }
        }
    }

    if (SPLIT) __syncthreads(); else __syncwarp();       // rr is dead from here on: its bytes become the staging rows
    // ---- angular (Eq. 5) ------------------------------------------------------------------------------
    static_assert(NAg * NZg == 32 && NAg + NZg == 12, "angular grid");
    const int za = lane % NZg, aa = lane / NZg;          // this lane's feature (a, z) of a pair block, index NZg a + z
    float facc = 0.f;                                    // running sum of feature (aa, za) of the current pair
    int e = 0;                                           // table entry of this lane's slot (monotonic over the rounds)
    for (int T0 = 32 * sw; T0 < T_pad; T0 += 32 * NWARP) {
        const int t = T0 + lane;
        float A[NZg], B[NAg];
#pragma unroll
        for (int z = 0; z < NZg; ++z) A[z] = 0.f;
#pragma unroll
        for (int a = 0; a < NAg; ++a) B[a] = 0.f;
        int my_blk = 0;                                  // angular block of this lane's slot
        bool my_end = false;                             // this slot is the last one of its species pair
        if (t < T_pad) {
            int next = S.tab[e + 1].x;
            while (t >= next) { ++e; next = S.tab[e + 1].x; }
            const int4 E = S.tab[e];
            my_blk = E.w;
            my_end = t + 1 == next;
            const int u = t - E.x;
            if (u < E.z) {
                // u -> (x, y) with u = x nk + y.  Different species: j = j0 + x, k = k0 + y.  Same species: distance
                // enumeration of the unordered pairs of nk items (d = x, j = y, k = y + d + 1 mod nk), each pair once.
                const int j0 = E.y & 255, k0 = (E.y >> 8) & 255, nk = (E.y >> 16) & 255;
                int x = (int)(((float)u + 0.5f) * fast_rcp((float)nk));
                int y = u - x * nk;
                if (y < 0) { --x; y += nk; } else if (y >= nk) { ++x; y -= nk; }
                int j, k;
                if (!(E.y >> 24)) { j = j0 + x; k = k0 + y; }
                else { j = j0 + y; k = y + x + 1; if (k >= nk) k -= nk; k += j0; }
                const float4 qj = S.nb[j], qk = S.nb[k];
                const float c = qj.x * qk.x + qj.y * qk.y + qj.z * qk.z;
                const float cx = qj.y * qk.z - qj.z * qk.y, cy = qj.z * qk.x - qj.x * qk.z, cz = qj.x * qk.y - qj.y * qk.x;
                const float sn = fast_sqrt(cx * cx + cy * cy + cz * cz);
                const float f2 = 2.0f * S.fca[j] * S.fca[k];
                const float Rm = 0.5f * (qj.w + qk.w);
#pragma unroll
                for (int z = 0; z < NZg; ++z) {
                    const float uu = fmaxf(fmaf(0.5f * K.sin_z[z], sn, fmaf(0.5f * K.cos_z[z], c, 0.5f)), 0.f);
                    A[z] = (AEV_ABL & 4) ? f2 * uu : f2 * fast_exp2(K.zeta * fast_log2(uu));    // 2 ((1+cos(theta-theta_z))/2)^zeta f_j f_k
                }
#pragma unroll
                for (int a = 0; a < NAg; ++a) {
                    const float mm = Rm - K.shf_a[a];
                    B[a] = (AEV_ABL & 4) ? mm : fast_exp2(-K.eta_a_l2e * mm * mm);
                }
            }
        }
#pragma unroll
        for (int z = 0; z < NZg; ++z) Sw.st[z][lane] = A[z];
#pragma unroll
        for (int a = 0; a < NAg; ++a) Sw.st[NZg + a][lane] = B[a];
        __syncwarp();
        // phase 2: the 8 quads of the round in order (pairs are padded to whole quads, so a pair ends at a quad end);
        // the branch is warp-uniform
        const unsigned endmask = __ballot_sync(FULL, my_end);
#pragma unroll
        for (int qd = 0; qd < ((AEV_ABL & 2) ? 0 : 8); ++qd) {
            const float4 a4 = *reinterpret_cast<const float4*>(&Sw.st[za][4 * qd]);
            const float4 b4 = *reinterpret_cast<const float4*>(&Sw.st[NZg + aa][4 * qd]);
            facc = fmaf(a4.x, b4.x, facc); facc = fmaf(a4.y, b4.y, facc);
            facc = fmaf(a4.z, b4.z, facc); facc = fmaf(a4.w, b4.w, facc);
            if ((endmask >> (4 * qd + 3)) & 1u) {             // pair complete: its 32 features go out, 64 (128) contiguous bytes
                const int blk = __shfl_sync(FULL, my_blk, 4 * qd + 3);
                if (SPLIT) part[blk * 32 + lane] += facc; else PUT_ANG(facc, blk);
                facc = 0.f;
            }
        }
        if (SPLIT) {                                         // this warp's next round is NWARP rounds away: bank the open pair's partial sum
            const int blk = __shfl_sync(FULL, my_blk, 31);
            part[blk * 32 + lane] += facc;
            facc = 0.f;
        }
        __syncwarp();
    }
    __syncwarp();
    if (SPLIT) {
        __syncthreads();
        const float* all = reinterpret_cast<const float*>(smem_raw + sizeof(WarpSmemFwd) * AEV_WARPS);
        for (int p = w; p < NPAIR; p += AEV_WARPS) {
            if (!((nz_pairs >> p) & 1u)) continue;
            float v = 0.f;
#pragma unroll
            for (int q = 0; q < AEV_WARPS; ++q) v += all[(size_t)q * (NPAIR * 32) + p * 32 + lane];
            PUT_ANG(v, p);
        }
        if (w != 0) return;                                  // the zeros below are warp 0's
    }

    // ---- zeros for what this atom lacks but a reader will touch -------------------------------------------
    // (tensor path: the feature blocks that are active for the row's tile; fp32 rows: everything)
    unsigned mask = 0xffffu;
    if (PLANES) { mask = tile_mask[row / ROW_TILE]; if (mask == 0) mask = 1u << 14; }   // G1 runs one zero block for an all-zero tile
    // lane p < 28: angular block p is read (its 64-wide block is active) but this atom has no such pair
    unsigned zm = __ballot_sync(FULL, lane < NPAIR && ((mask >> (lane >> 1)) & 1u) && !((nz_pairs >> lane) & 1u));
    for (; zm; zm &= zm - 1u) PUT_ANG(0.f, __ffs(zm) - 1);
    // lane q < 8: radial slot q (priority order; slot 7 is the 16 padding columns) likewise
    bool rz = false;
    if (lane < 8) {
        bool absent = true;
        if (lane < NSP) {
            const int s = prio_sp(lane);
            absent = nst == 0 || seg_cnt[(size_t)i * 16 + s] + seg_cnt[(size_t)i * 16 + 8 + s] == 0;
        }
        rz = absent && ((mask >> (14 + (lane >> 2))) & 1u);
    }
    unsigned rm = __ballot_sync(FULL, rz);
    for (; rm; rm &= rm - 1u)
        if (lane < 16) PUT_RAD(0.f, __ffs(rm) - 1);
}

// -------------------------------------------------------------------------------------------------
// backward (a5): F = -sum_i sum_m dE/dG_i[m] dG_i[m]/dr, one warp per central atom i
//   neighbours   lane <-> neighbour (rounds of 32): geometry once, the whole radial derivative of that neighbour
//                (16 shifts) in registers; the lane keeps the force of "its" neighbours (slots lane, lane+32, lane+64)
//                in registers until the end.
//   angular      triplets in distance order, t = d na + j, k = j + d + 1 (mod na): lane <-> triplet computes the two
//                gradient vectors (on j and on k) and stages them; then lane <-> neighbour n gathers the (at most
//                two per distance d present in the round) staged vectors that belong to n - closed-form slot
//                indices, so there are no atomics and no read-modify-write in shared memory.
//   scatter      one global atomic triple per neighbour and one for the centre.
// -------------------------------------------------------------------------------------------------
#ifndef BWD_W
#define BWD_W 8
#endif
constexpr int BWD_WARPS = BWD_W;
#ifndef BWD_MINB
#define BWD_MINB (32 / BWD_W)
#endif

constexpr int OWN = 3;   // neighbour slots per lane that can be angular (MAX_ANG = 96 = 3 x 32)
static_assert(MAX_ANG <= OWN * 32, "angular neighbours must fit the per-lane force registers");

struct __align__(16) WarpSmemBwd {
    float g_rad[NSP * NR];       // radial blocks by neighbour species
    float4 nb[MAX_ANG];          // ux, uy, uz, R of the angular neighbours
    float2 fd[MAX_ANG];          // f_c(R; Rca), f_c'(R; Rca)
    float st[6][32];             // staged gradient vectors of one round: on j (x, y, z), on k (x, y, z)
    int sp[MAX_ANG];
};

// SPLIT (small systems): one block of 8 warps per atom - warp 0 does the neighbour pass, the angular rounds are dealt out to the
// 8 warps (one warp per atom is latency-bound: ~4 k dependent instructions, 36 us for a 50-atom solute whatever its size)
template <int NAg, int NZg, bool SPLIT>
__global__ void __launch_bounds__(BWD_WARPS * 32, BWD_MINB)
k_aev_bwd(const float4* __restrict__ spos, const int* __restrict__ row_ptr, const int* __restrict__ col,
          const unsigned short* __restrict__ seg_cnt, const int* __restrict__ rowmap, const Grid* __restrict__ gp,
          const __grid_constant__ AevConst K, int n, const float* __restrict__ grad, float* __restrict__ fsorted,
          const int* __restrict__ row_slot) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ Grid g;
    if (threadIdx.x == 0) g = *gp;
    __syncthreads();
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int i = SPLIT ? (int)blockIdx.x : blockIdx.x * BWD_WARPS + w;   // warp <-> atom (SPLIT: block <-> atom), or <-> row in a partial evaluation
    if (i >= n) return;
    if (row_slot) { i = row_slot[i]; if (i < 0) return; }
    WarpSmemBwd& S = reinterpret_cast<WarpSmemBwd*>(smem_raw)[SPLIT ? 0 : w];     // geometry of the atom's neighbours
    WarpSmemBwd& Sw = reinterpret_cast<WarpSmemBwd*>(smem_raw)[w];                 // this warp's staging rows
    const int sw = SPLIT ? w : 0;                                                  // this warp's share of the angular rounds
    constexpr int NWARP = SPLIT ? BWD_WARPS : 1;
    const unsigned FULL = 0xffffffffu;

    // run lengths of the row (as in the forward kernel)
    int cnt = (lane < 16 && lane != 7 && lane != 15) ? (int)seg_cnt[(size_t)i * 16 + lane] : 0;
    int start = cnt;
#pragma unroll
    for (int o = 1; o < 16; o <<= 1) {
        int y = __shfl_up_sync(FULL, start, o);
        if (lane >= o) start += y;
    }
    start -= cnt;
    int na = __shfl_sync(FULL, start, 8);
    int nst = __shfl_sync(FULL, start, 15);
    if (na > MAX_ANG || nst > MAX_RAD) { na = 0; nst = 0; cnt = 0; }     // capacity overflow: reported by the forward pass

    // ---- the blocks of dE/dG this atom uses ----------------------------------------------------------------
    const int row_i = rowmap[i];
    if (row_i < 0) return;                             // not a central atom of this call (partial evaluation)
    const float* grow = grad + (size_t)row_i * AEV_LD;
    // The neighbour chain (row_ptr -> col -> spos) and the dE/dG rows (DRAM) are independent: request the first two
    // rounds of neighbours now, so that their latency runs under the staging of the gradient blocks below
    const int rb = row_ptr[i];
    const float4 pi = spos[i];
    constexpr int PRE = 2;
    int jg_pre[PRE];
    float4 pj_pre[PRE];
#pragma unroll
    for (int q = 0; q < PRE; ++q) {
        const int a = lane + 32 * q;
        jg_pre[q] = a < nst ? col[rb + a] : i;
    }
#pragma unroll
    for (int q = 0; q < PRE; ++q) pj_pre[q] = spos[jg_pre[q]];
    {
        int psa = 0, psb = 0;
        if (lane < NPAIR) { const int e = c_pair_sp[lane]; psa = e & 15; psb = e >> 4; }
        const int ca = __shfl_sync(FULL, cnt, psa), cb = __shfl_sync(FULL, cnt, psb);
        // the angular blocks of dE/dG are read straight from the row (4 KB, L1-resident after the first touch): no staging
        // copy, and 4 KB less shared memory per warp (occupancy); touch the blocks this atom uses now so the lines arrive early
        unsigned nz = __ballot_sync(FULL, lane < NPAIR && ((psa == psb) ? ca > 1 : (ca > 0 && cb > 0)));
        for (; nz; nz &= nz - 1u) {
            const int p = __ffs(nz) - 1;
            asm volatile("prefetch.global.L1 [%0];" ::"l"(grow + 32 * p + (lane & 1) * 16));
        }
        for (int s = 0; s < NSP; ++s)
            if (__shfl_sync(FULL, cnt, s) + __shfl_sync(FULL, cnt, 8 + s) > 0 && lane < NR && sw == 0) S.g_rad[NR * s + lane] = grow[rad_col(s) + lane];
    }
    __syncwarp();

    const float inv_rcr = 1.0f / K.rcr, inv_rca = 1.0f / K.rca;
    float fix = 0.f, fiy = 0.f, fiz = 0.f;              // force on the centre, summed over this lane's terms
    float Fx[OWN], Fy[OWN], Fz[OWN];                    // forces on the neighbours lane, lane + 32, lane + 64
    int cj[OWN];
#pragma unroll
    for (int q = 0; q < OWN; ++q) { Fx[q] = Fy[q] = Fz[q] = 0.f; cj[q] = 0; }

    // ---- neighbours: geometry, staging of the angular ones, radial derivative (Eq. 4) -----------------------
#pragma unroll
    for (int q = 0; q < MAX_RAD / 32; ++q) {
        const int a = lane + 32 * q;
        if (SPLIT && sw != 0) {                              // the neighbour pass is warp 0's; the others only need the slots
            if (q < OWN && a < nst) cj[q] = q < PRE ? jg_pre[q < PRE ? q : 0] : col[rb + a];
        } else if (32 * q < nst && a < nst) {
            const int jg = q < PRE ? jg_pre[q < PRE ? q : 0] : col[rb + a];
            const NbrGeom nbq = neighbour_geom(pi, q < PRE ? pj_pre[q < PRE ? q : 0] : spos[jg], g);
            const float fc = fcut(nbq.R, inv_rcr), dfc = dfcut(nbq.R, inv_rcr, K.pi_over_rcr);
            const float c1 = -2.0f * K.eta_r * fc;
            const float4* gr = reinterpret_cast<const float4*>(&S.g_rad[NR * nbq.sp]);
            float coef = 0.f;
#pragma unroll
            for (int m4 = 0; m4 < ((AEV_ABL & 16) ? 0 : NR / 4); ++m4) {
                const float4 g4 = gr[m4];
                const float gm[4] = {g4.x, g4.y, g4.z, g4.w};
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const float dr = nbq.R - K.shf_r[4 * m4 + e];
                    const float t = fast_exp2(-K.eta_r_l2e * dr * dr);
                    coef = fmaf(gm[e] * t, fmaf(c1, dr, dfc), coef);
                }
            }
            const float vx = coef * nbq.ux, vy = coef * nbq.uy, vz = coef * nbq.uz;
            fix += vx; fiy += vy; fiz += vz;
            if (a < na) {
                S.nb[a] = make_float4(nbq.ux, nbq.uy, nbq.uz, nbq.R);
                S.fd[a] = make_float2(fcut(nbq.R, inv_rca), dfcut(nbq.R, inv_rca, K.pi_over_rca));
                S.sp[a] = nbq.sp;
            }
            if (q < OWN) { Fx[q] = -vx; Fy[q] = -vy; Fz[q] = -vz; cj[q] = jg; }
            else {
                atomicAdd(&fsorted[3 * jg + 0], -vx);
                atomicAdd(&fsorted[3 * jg + 1], -vy);
                atomicAdd(&fsorted[3 * jg + 2], -vz);
            }
        }
    }
    if (SPLIT) __syncthreads(); else __syncwarp();

    // ---- angular (Eq. 5) -----------------------------------------------------------------------------------
    const int npairs = na * (na - 1) / 2;
    const float inv_na = na > 0 ? fast_rcp((float)na) : 0.f;
    // distance of the round's first and last slot, carried from round to round (T0 = d0 na + r0; an integer division per round
    // was 6 % of the kernel's instructions)
    int d0 = 0, r0 = 32 * sw;
    while (na > 0 && r0 >= na) { r0 -= na; ++d0; }
    for (int T0 = 32 * sw; T0 < ((AEV_ABL & 128) ? 0 : npairs); T0 += 32 * NWARP) {
        const int t = T0 + lane;
        if (t < npairs) {
            int d = (int)(((float)t + 0.5f) * inv_na);
            int j = t - d * na;
            if (j < 0) { --d; j += na; } else if (j >= na) { ++d; j -= na; }
            int k = j + d + 1;
            if (k >= na) k -= na;
            const float4 qj = S.nb[j], qk = S.nb[k];
            const float2 fj = S.fd[j], fk = S.fd[k];
            const float c = qj.x * qk.x + qj.y * qk.y + qj.z * qk.z;
            const float cx = qj.y * qk.z - qj.z * qk.y, cy = qj.z * qk.x - qj.x * qk.z, cz = qj.x * qk.y - qj.y * qk.x;
            const float sn = fast_sqrt(cx * cx + cy * cy + cz * cz);
            const float Rm = 0.5f * (qj.w + qk.w);
            const float4* gb = reinterpret_cast<const float4*>(grow + 32 * ipair(S.sp[j], S.sp[k]));
            f32x2 AdA[NZg];                                                        // (A_z, dA_z/dtheta) as packed pairs
#pragma unroll
            for (int z = 0; z < NZg; ++z) {
                const float u = fmaxf(fmaf(0.5f * K.sin_z[z], sn, fmaf(0.5f * K.cos_z[z], c, 0.5f)), 0.f);
                const float wz = fast_exp2((K.zeta - 1.0f) * fast_log2(u));       // u^(zeta-1)
                AdA[z] = pack2(2.0f * u * wz,                                      // A = 2 u^zeta
                               -K.zeta * wz * (sn * K.cos_z[z] - c * K.sin_z[z])); // dA/dtheta
            }
            f32x2 S0t = pack2(0.f, 0.f);                                           // (S0, St)
            float Sm = 0.f;
#pragma unroll
            for (int a = 0; a < ((AEV_ABL & 32) ? 0 : NAg); ++a) {
                const float mm = Rm - K.shf_a[a];
                const float B = fast_exp2(-K.eta_a_l2e * mm * mm);
                const float dB = -K.eta_a * mm * B;                                // dB/dR_ij = dB/dR_ik
                f32x2 uv = pack2(0.f, 0.f);                                        // (ua, va) over the entries (a, z) of the pair block: [a][z]
#pragma unroll
                for (int z4 = 0; z4 < NZg / 4; ++z4) {
                    const float4 g4 = __ldg(gb + a * (NZg / 4) + z4);
                    uv = fma2(pack2(g4.x, g4.x), AdA[4 * z4], uv);
                    uv = fma2(pack2(g4.y, g4.y), AdA[4 * z4 + 1], uv);
                    uv = fma2(pack2(g4.z, g4.z), AdA[4 * z4 + 2], uv);
                    uv = fma2(pack2(g4.w, g4.w), AdA[4 * z4 + 3], uv);
                }
                S0t = fma2(pack2(B, B), uv, S0t);
                float ua, va;
                unpack2(uv, ua, va);
                Sm = fmaf(dB, ua, Sm);
            }
            float S0, St;
            unpack2(S0t, S0, St);
            const float dth = St * fj.x * fk.x;                                    // sum g dT/dtheta
            const float dRj = (Sm * fj.x + S0 * fj.y) * fk.x;                      // sum g dT/dR_ij
            const float dRk = (Sm * fk.x + S0 * fk.y) * fj.x;
            const float inv_s = sn > 1e-20f ? fast_rcp(sn) : 0.f;                  // collinear: e = 0 (Q7)
            const float tj = -dth * inv_s * fast_rcp(qj.w), tk = -dth * inv_s * fast_rcp(qk.w);   // d theta/d r_j = -e_j / R_ij
            const float gjx = tj * (qk.x - c * qj.x) + dRj * qj.x, gjy = tj * (qk.y - c * qj.y) + dRj * qj.y,
                        gjz = tj * (qk.z - c * qj.z) + dRj * qj.z;
            const float gkx = tk * (qj.x - c * qk.x) + dRk * qk.x, gky = tk * (qj.y - c * qk.y) + dRk * qk.y,
                        gkz = tk * (qj.z - c * qk.z) + dRk * qk.z;
            fix += gjx + gkx; fiy += gjy + gky; fiz += gjz + gkz;
            Sw.st[0][lane] = gjx; Sw.st[1][lane] = gjy; Sw.st[2][lane] = gjz;
            Sw.st[3][lane] = gkx; Sw.st[4][lane] = gky; Sw.st[5][lane] = gkz;
        }
        __syncwarp();
        // gather: neighbour nn is j of slot d na + nn and k of slot d na + (nn - d - 1 mod na), for every d in the round
        const int cntr = min(32, npairs - T0);
        const int d_lo = d0;
        int d_hi = d0, rl = r0 + cntr - 1;
        while (rl >= na) { rl -= na; ++d_hi; }
#pragma unroll
        for (int q = 0; q < OWN; ++q) {
            const int nn = lane + 32 * q;
            if (32 * q < na && nn < na && !(AEV_ABL & 64)) {
                for (int d = d_lo; d <= d_hi; ++d) {
                    const int tj = d * na + nn - T0;
                    if ((unsigned)tj < (unsigned)cntr) { Fx[q] -= Sw.st[0][tj]; Fy[q] -= Sw.st[1][tj]; Fz[q] -= Sw.st[2][tj]; }
                    int jj = nn - d - 1;
                    if (jj < 0) jj += na;
                    const int tk = d * na + jj - T0;
                    if ((unsigned)tk < (unsigned)cntr) { Fx[q] -= Sw.st[3][tk]; Fy[q] -= Sw.st[4][tk]; Fz[q] -= Sw.st[5][tk]; }
                }
            }
        }
        r0 += 32 * NWARP;
        while (r0 >= na) { r0 -= na; ++d0; }
        __syncwarp();
    }

    // ---- scatter ---------------------------------------------------------------------------------------------
#pragma unroll
    for (int q = 0; q < OWN; ++q) {
        if (lane + 32 * q < nst) {
            atomicAdd(&fsorted[3 * cj[q] + 0], Fx[q]);
            atomicAdd(&fsorted[3 * cj[q] + 1], Fy[q]);
            atomicAdd(&fsorted[3 * cj[q] + 2], Fz[q]);
        }
    }
    for (int o = 16; o; o >>= 1) {
        fix += __shfl_xor_sync(FULL, fix, o);
        fiy += __shfl_xor_sync(FULL, fiy, o);
        fiz += __shfl_xor_sync(FULL, fiz, o);
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
                                double* __restrict__ E, const int* __restrict__ status, int* __restrict__ sticky) {
    __shared__ double part[32];
    // every kernel that can raise a data-dependent fault has run by now: fold the call's status word into the sticky one
    if (blockIdx.x == 0 && threadIdx.x == 0) { const int s = *status; if (s != 0) atomicCAS(sticky, 0, s); }
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
// per-device kernel attributes (dynamic shared memory above 48 KB); called once per context from dhp_create
int aev_init(Ctx* ctx) {
    for (int hi = 0, p = 0; hi < NSP; ++hi)            // the literal table above must match prio_sp()
        for (int lo = 0; lo <= hi; ++lo, ++p)
            if ((prio_sp(lo) | (prio_sp(hi) << 4)) != (int)h_pair_sp[p]) return DHP_E_BADARG;
    const int fs = (int)(sizeof(WarpSmemFwd) * AEV_WARPS), bs = (int)(sizeof(WarpSmemBwd) * BWD_WARPS);
    const int fss = fs + (int)(sizeof(float) * AEV_WARPS * NPAIR * 32);      // SPLIT: + the warps' pair-block sums
    DHP_CUDA(ctx, cudaFuncSetAttribute((k_aev_fwd<false, 8, 4, false>), cudaFuncAttributeMaxDynamicSharedMemorySize, fs));
    DHP_CUDA(ctx, cudaFuncSetAttribute((k_aev_fwd<true, 8, 4, false>), cudaFuncAttributeMaxDynamicSharedMemorySize, fs));
    DHP_CUDA(ctx, cudaFuncSetAttribute((k_aev_fwd<false, 4, 8, false>), cudaFuncAttributeMaxDynamicSharedMemorySize, fs));
    DHP_CUDA(ctx, cudaFuncSetAttribute((k_aev_fwd<true, 4, 8, false>), cudaFuncAttributeMaxDynamicSharedMemorySize, fs));
    DHP_CUDA(ctx, cudaFuncSetAttribute((k_aev_fwd<false, 8, 4, true>), cudaFuncAttributeMaxDynamicSharedMemorySize, fss));
    DHP_CUDA(ctx, cudaFuncSetAttribute((k_aev_fwd<true, 8, 4, true>), cudaFuncAttributeMaxDynamicSharedMemorySize, fss));
    DHP_CUDA(ctx, cudaFuncSetAttribute((k_aev_fwd<false, 4, 8, true>), cudaFuncAttributeMaxDynamicSharedMemorySize, fss));
    DHP_CUDA(ctx, cudaFuncSetAttribute((k_aev_fwd<true, 4, 8, true>), cudaFuncAttributeMaxDynamicSharedMemorySize, fss));
    DHP_CUDA(ctx, cudaFuncSetAttribute((k_aev_bwd<8, 4, false>), cudaFuncAttributeMaxDynamicSharedMemorySize, bs));
    DHP_CUDA(ctx, cudaFuncSetAttribute((k_aev_bwd<4, 8, false>), cudaFuncAttributeMaxDynamicSharedMemorySize, bs));
    DHP_CUDA(ctx, cudaFuncSetAttribute((k_aev_bwd<8, 4, true>), cudaFuncAttributeMaxDynamicSharedMemorySize, bs));
    DHP_CUDA(ctx, cudaFuncSetAttribute((k_aev_bwd<4, 8, true>), cudaFuncAttributeMaxDynamicSharedMemorySize, bs));
    return DHP_OK;
}

int aev_forward(Ctx* ctx, bool planes) {
    const int n = (int)ctx->n_atoms;
    ctx->aev_in_planes = planes;
    if (n == 0) return DHP_OK;
    const size_t smem = sizeof(WarpSmemFwd) * AEV_WARPS;
    // partial evaluation: one warp per ROW; the host knows an upper bound of the row count only when it knows the number
    // of central atoms, which it does not (the mask lives on the device) - the row tables are walked up to max_rows of the
    // call's atom count instead, and rows beyond the last group hold -1
    const int* row_slot = ctx->partial ? ctx->row_slot : nullptr;
    const int nw = ctx->partial ? (int)std::min<int64_t>(ctx->max_rows, (int64_t)n + NSP * ROW_ALIGN) : n;
    // small systems: a block of 8 warps per atom (SPLIT), else a warp per atom
    const bool split = n <= SMALL_N && !ctx->no_fwd_split;      // measured: 50 atoms 26.7 -> 14.6 us, 288 atoms 15.1 -> 12.6 us
    const int blocks = split ? nw : (nw + AEV_WARPS - 1) / AEV_WARPS;
    const size_t smem_l = smem + (split ? sizeof(float) * AEV_WARPS * NPAIR * 32 : 0);
    const size_t plane_stride = (size_t)ctx->max_rows * AEV_LD;
#define DHP_AEV_FWD(P, A, Z, S)                                                                                                 \
    DHP_LAUNCH(ctx, (k_aev_fwd<P, A, Z, S>), blocks, AEV_WARPS * 32, smem_l, ctx->spos, ctx->row_ptr, ctx->col, ctx->seg_cnt, ctx->rowmap, \
               ctx->tile_mask, ctx->grid, ctx->aevc, nw, ctx->aev, ctx->aev_planes, plane_stride, ctx->status, row_slot)
    const bool g84 = ctx->aevc.n_a == 8;                 // 8 x 4 (ANI-2x shape) or 4 x 8 (ANI-1x shape) angular grid
    if (split) {
        if (planes) { if (g84) DHP_AEV_FWD(true, 8, 4, true); else DHP_AEV_FWD(true, 4, 8, true); }
        else        { if (g84) DHP_AEV_FWD(false, 8, 4, true); else DHP_AEV_FWD(false, 4, 8, true); }
    } else {
        if (planes) { if (g84) DHP_AEV_FWD(true, 8, 4, false); else DHP_AEV_FWD(true, 4, 8, false); }
        else        { if (g84) DHP_AEV_FWD(false, 8, 4, false); else DHP_AEV_FWD(false, 4, 8, false); }
    }
#undef DHP_AEV_FWD
    DHP_CUDA(ctx, cudaGetLastError());
    return DHP_OK;
}

int aev_backward(Ctx* ctx, float* F_out) {
    const int n = (int)ctx->n_atoms;
    if (n == 0) return DHP_OK;
    const size_t smem = sizeof(WarpSmemBwd) * BWD_WARPS;
    // fsorted was zeroed with the rest of the per-call arena at the start of the call (nlist_build)
    const int* row_slot = ctx->partial ? ctx->row_slot : nullptr;
    const int nw = ctx->partial ? (int)std::min<int64_t>(ctx->max_rows, (int64_t)n + NSP * ROW_ALIGN) : n;
    // small systems: a block of 8 warps per atom (SPLIT), else a warp per atom
    const bool split = n <= 128;                       // measured: 50 atoms 44 -> 23 us; at 288 atoms a warp per atom is faster (19 vs 40 us)
    const int blocks = split ? nw : (nw + BWD_WARPS - 1) / BWD_WARPS;
#define DHP_AEV_BWD(A, Z, S)                                                                                                  \
    DHP_LAUNCH(ctx, (k_aev_bwd<A, Z, S>), blocks, BWD_WARPS * 32, smem, ctx->spos, ctx->row_ptr, ctx->col, ctx->seg_cnt, ctx->rowmap, \
               ctx->grid, ctx->aevc, nw, ctx->grad, ctx->fsorted, row_slot)
    if (ctx->aevc.n_a == 8) { if (split) DHP_AEV_BWD(8, 4, true); else DHP_AEV_BWD(8, 4, false); }
    else                    { if (split) DHP_AEV_BWD(4, 8, true); else DHP_AEV_BWD(4, 8, false); }
#undef DHP_AEV_BWD
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
    DHP_LAUNCH(ctx, k_energy_reduce, blocks, 256, 0, ctx->e_atom, ctx->row_slot, ctx->smol, ctx->sp_start, per_mol, E_out, ctx->status, ctx->sticky);
    DHP_CUDA(ctx, cudaGetLastError());
    return DHP_OK;
}

}  // namespace dhp
