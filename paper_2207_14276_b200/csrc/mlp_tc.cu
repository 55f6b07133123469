// a3 + a4 on the 5th-generation tensor cores: tcgen05.mma with TMEM accumulators, operands staged by TMA
// (Eq. 2, L159 ensemble, L161 "back-propagation" = the dominant cost).
//
// Arithmetic.  Single-pass fp16/bf16/tf32 misses the force tolerance by an order of magnitude,
// so every operand x is kept as a two-term fp16 split  x = hi + lo  (hi = fp16(x), lo = fp16(x - hi)) and every
// product is three MMAs into the same fp32 accumulator:  hi*hi + hi*lo + lo*hi  (the dropped lo*lo term is
// 2^-22 relative).  Weights are pre-scaled by 2^6 and back-propagated deltas by 2^10 so that the lo terms stay in
// the fp16 normal range; the power-of-two scales are removed exactly in the epilogues.
//
// Activation layout.  An epilogue thread owns one row (one TMEM lane), so row-major activations make every
// 16-byte store of a warp land in a different 128-byte line.  The activation planes (h1, h2, d3, d2, d1) are
// therefore stored as the image of the no-swizzle K-major UMMA operand tile:
//     [plane hi/lo][row tile][64-column block][8-column group (8)][row in tile (128)][8 halves = 16 B]
// so that the 32 lanes of a warp write (and, for CELU', read back) 512 contiguous bytes per instruction, and the
// next GEMM fetches its A operand as one contiguous 16 KB cp.async.bulk per plane and K block (descriptor:
// SWIZZLE_NONE, leading byte offset 2048 = next 8-column group, stride byte offset 128 = next 8 rows).
// The AEV planes (A of G1) are written in the same tiled layout by the AEV kernel (aev_tiled_off()); the weights (B) of
// k_gemm_tc / k_gemm_tc2 stay row-major and come in through TMA tensor maps with SWIZZLE_128B, those of the
// chain kernels (k_mlp_fused, k_mlp_mid) are pre-tiled images fetched with plain bulk copies.
//
// Default path (two launches): k_mlp_fused = G1 + G2 + G3 + output layer + B3 + B2 for one (row tile, network) per work item,
// every intermediate on chip (further down), then B1 = k_gemm_tc2.  The persistent, warp-specialised template below runs any
// one of the six GEMMs as its own launch: B1, the two-launch path (DHP_TC_FUSE=0: G1, then k_mlp_mid), the layer-by-layer mode:
//   warps 0..7  epilogue       (tcgen05.ld 32x32b -> bias / CELU / CELU' / split -> global), overlapped with the
//                               next tile's MMAs through two TMEM accumulator stages (2 x 256 columns)
//   warp 8      TMA producer   (cp.async.bulk.tensor.2d, SWIZZLE_128B, 64-wide K blocks, mbarrier ring)
//   warp 9      MMA issuer     (one elected lane: 3 x tcgen05.mma.cta_group::1.kind::f16 per 16-wide K step)
// The two single-thread roles take the HIGHEST warp ids: the warp scheduler of an SM sub-partition serves the highest
// eligible warp id first, and an MMA issuer that loses its issue slots to the epilogue warps stalls the tensor pipe.
// Tile = 128 rows (atoms of ONE species: row groups start at multiples of 128) x BN columns; tiles of the same
// row block are adjacent in the schedule so that concurrently running CTAs share the A tile through L2.
//
//   G1  H1 = CELU(G W1^T + b1)          K = 1024 (1008 padded)  BN = 256  n-tiles = models
//   G2  H2 = CELU(H1 W2^T + b2)         K = 256                 BN = 192
//   G3  H3 = CELU(H2 W3^T + b3);  E_i += (w4.H3 + b4)/M;  D3 = w4 * CELU'(z3) / M      K = 192, BN = 160
//   B3  D2 = (D3 W3) * CELU'(z2)        K = 160                 BN = 192
//   B2  D1 = (D2 W2) * CELU'(z1)        K = 192                 BN = 256
//   B1  dE/dG = sum_e D1_e W1_e         K = models*256          BN = 256  n-tiles = 4
#include <cuda.h>
#include <cuda_fp16.h>
#include <new>
#include <stdio.h>
#include <string.h>

#include "dhp_internal.cuh"

namespace dhp {

namespace {

constexpr int BM = 128;            // rows per tile (UMMA M)
constexpr int BK = 64;             // K elements per stage (128 bytes of fp16: one SWIZZLE_128B row)
constexpr int STAGES = 2;
constexpr int A_PLANE_BYTES = BM * BK * 2;       // 16 KB
constexpr int B_SLOT_BYTES = 256 * BK * 2;       // 32 KB (BN <= 256)
constexpr int STAGE_BYTES = 2 * A_PLANE_BYTES + 2 * B_SLOT_BYTES;   // 96 KB
constexpr int OUT_STAGE_BYTES = 2 * BM * KBLK * 2;     // one 64-column block of a tiled activation output, hi plane then lo plane (32 KB)
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + OUT_STAGE_BYTES + 1024 /*align*/ + 256 /*barriers, TMEM word, tile ring*/;
constexpr int TMEM_COLS = 512;
constexpr int ACC_STRIDE = 256;    // TMEM columns per accumulator stage
constexpr int EPI_WARPS = 8;         // two per TMEM lane quadrant, splitting the column chunks
constexpr int RING = 4;              // depth of the tile-id ring between the scheduler (TMA warp) and the other roles
constexpr int NB_BLOCK_BYTES = KBLK * BK * 2;   // one 64-row block of a B tile (8 KB)
constexpr int TC_THREADS = 64 + 32 * EPI_WARPS;
constexpr float W_SCALE = 64.0f;       // 2^6 on every weight matrix
constexpr float D_SCALE = 1024.0f;     // 2^10 on the back-propagated deltas

enum { EPI_CELU = 0, EPI_OUT = 1, EPI_DCELU = 2, EPI_GRAD = 3 };

struct TcArgs {
    int single;               // 1: single-pass fp16 (hi x hi only; opt-in mixed precision, DHP_MLP_TENSOR_FP16)
    int K;                    // reduction length in elements (multiple of 16)
    int BN;                   // tile width (multiple of 16, <= 256)
    int n_tiles;              // column tiles per row block
    int a_k_off_per_tile;     // A column offset per column tile (per-model activations), else 0
    int a_plane_rows;         // rows of one A plane (lo plane starts there)
    int b_rows_per_species;   // rows of one B plane of one species
    int b_rows_per_tile;      // B row offset per column tile
    float acc_scale;          // removes the power-of-two operand scales
    const int* row_species;
    const int* sp_start;
    const float* bias;        // [species][n_tiles*BN]  (EPI_CELU, EPI_OUT)
    const float* w4;          // [species][models*160]  (EPI_OUT)
    const float* b4;          // [species][models]
    float inv_models;
    float alpha;
    __half* out_planes;       // tiled activation planes (hi plane then lo plane)
    int out_ld;               // EPI_GRAD: row pitch of out_f32
    const __half* h_planes;   // saved activations for CELU' (EPI_DCELU), same geometry as out
    float* out_f32;           // EPI_GRAD: [rows][out_ld]
    float* e_atom;            // EPI_OUT
    const __half* a_tiled;    // A in the tiled activation layout (null: A comes through tmA, row-major AEV planes)
    int a_kblocks;            // 64-column blocks per row tile of the A buffer
    int a_kb_per_tile;        // A block offset per column tile (per-model activations), else 0
    int plane_tiles;          // row tiles per plane of every activation buffer (max_rows / 128)
    int out_kblocks;          // 64-column blocks per row tile of the output buffer (and of h_planes)
    int out_cols_per_tile;    // output column pitch per column tile (BN, or 192 for the 160-wide d3)
    const unsigned* tile_mask;  // [row tiles] active 64-wide feature blocks (G1: K blocks to visit, B1: N blocks to produce)
    int* sched;               // dynamic tile counter of this launch (zeroed by the host)
    int ksplit;               // EPI_GRAD only: the K blocks of a tile are split over this many work items (power of two
                              // <= KB) which add their partial results into out_f32 (zeroed by the host) - small systems,
                              // where one tile's 32 sequential K blocks would leave most SMs idle
};

// how the feature-block mask of a row tile is used
enum { CMP_NONE = 0, CMP_K = 1, CMP_N = 2 };

// ---- PTX wrappers ------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile("{\n\t.reg .pred P;\n\telect.sync _|P, 0xffffffff;\n\tselp.b32 %0, 1, 0, P;\n\t}" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred P;\n"
        "WAIT_LOOP:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 P, [%0], %1;\n\t"
        "@P bra DONE;\n\t"
        "bra WAIT_LOOP;\n"
        "DONE:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar) : "memory");
}
__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// shared -> global bulk copy (the TMA store path: whole lines leave the SM without passing through the LSU / L1 store path,
// which is what limits an epilogue that writes its 128 KB tile with per-thread 16-byte stores - profiles/r2b)
__device__ __forceinline__ void bulk_store(void* dst, uint32_t src, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void named_bar(int id, int threads) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory"); }
__device__ __forceinline__ void prefetch_tmap(const CUtensorMap* map) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_alloc(uint32_t smem_dst, uint32_t cols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t cols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
}
__device__ __forceinline__ void umma_f16(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld32_issue(uint32_t taddr, uint32_t (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
          "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
          "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// K-major, SWIZZLE_128B shared-memory matrix descriptor (sm_100 format): start address >> 4 in bits [0,14),
// stride byte offset (8 rows x 128 B = 1024) >> 4 in bits [32,46), version 1 in bits [46,48), layout type 2
// (SWIZZLE_128B) in bits [61,64).  The leading byte offset is unused for swizzled K-major operands.
__device__ __forceinline__ uint64_t make_smem_desc(uint32_t saddr) {
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFF) >> 4);
    d |= (uint64_t)(1024 >> 4) << 32;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)2 << 61;
    return d;
}
// K-major operand without swizzle, [8-column group][row][16 B]: leading byte offset (next core matrix along K) 2048,
// stride byte offset (next 8 rows) 128
__device__ __forceinline__ uint64_t make_smem_desc_tiled(uint32_t saddr) {
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFF) >> 4);
    d |= (uint64_t)(2048 >> 4) << 16;
    d |= (uint64_t)(128 >> 4) << 32;
    d |= (uint64_t)1 << 46;
    return d;
}
// instruction descriptor: D = f32, A = B = f16, both K-major, M = 128, N = bn
__device__ __forceinline__ uint32_t make_idesc(int bn) {
    return (1u << 4) | ((uint32_t)(bn >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);
}

// CELU(v) = v (v > 0), alpha (exp(v/alpha) - 1) otherwise; k = log2(e)/alpha.  ex2.approx has 2^-22 relative error,
// so the absolute error of the negative branch is <= alpha 2^-22 (2.4e-8 at alpha = 0.1), below fp32 eps of O(1) values.
__device__ __forceinline__ float fast_ex2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float celu_f(float v, float alpha, float k) {
    const float e = fmaf(alpha, fast_ex2(v * k), -alpha);      // e > v for every v; e < 0 iff v < 0
    return fmaxf(v, fminf(e, 0.f));
}
// CELU'(z) from h = CELU(z): 1 for h > 0, h / alpha + 1 (<= 1) otherwise
__device__ __forceinline__ float dcelu_from_h(float h, float inv_alpha) { return fminf(fmaf(h, inv_alpha, 1.0f), 1.0f); }

// Blackwell's packed fp32 instructions (FFMA2 / FMUL2 / FADD2: two fp32 results per issue slot); the epilogues are bound by
// instruction issue (4 epilogue warps per scheduler, ~175 instructions per 16 columns), and rounding is that of the scalar forms
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float a, float b) { f32x2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void unpack2(f32x2 v, float& a, float& b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) { f32x2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) { f32x2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) { f32x2 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }

// two floats -> packed fp16 pair, round-to-nearest, saturating to the largest finite fp16 (first argument -> low half)
__device__ __forceinline__ uint32_t cvt_pack(float lo_half, float hi_half) {
    uint32_t r;
    asm("cvt.rn.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi_half), "f"(lo_half));
    return r;
}
// x = hi + lo for two values at once: hi = fp16(x), lo = fp16(x - hi)
__device__ __forceinline__ void split_pair(float x0, float x1, uint32_t& hi, uint32_t& lo) {
    hi = cvt_pack(x0, x1);
    const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&hi));
    float d0, d1;
    unpack2(sub2(pack2(x0, x1), pack2(f.x, f.y)), d0, d1);
    lo = cvt_pack(d0, d1);
}
__device__ __forceinline__ void split_half(float x, __half& hi, __half& lo) {
    x = fminf(fmaxf(x, -65000.f), 65000.f);
    hi = __float2half_rn(x);
    lo = __float2half_rn(x - __half2float(hi));
}

__device__ __forceinline__ uint32_t pack_half2(__half a, __half b) {
    __half2 h = __halves2half2(a, b);
    return *reinterpret_cast<uint32_t*>(&h);
}
__device__ __forceinline__ void unpack_add(uint32_t h, uint32_t l, float& a, float& b) {
    const float2 fh = __half22float2(*reinterpret_cast<__half2*>(&h));
    const float2 fl = __half22float2(*reinterpret_cast<__half2*>(&l));
    unpack2(add2(pack2(fh.x, fh.y), pack2(fl.x, fl.y)), a, b);
}
// 16 accumulator columns -> CELU(acc * sc + bias): the multiply-adds as packed pairs (same roundings as celu_f)
__device__ __forceinline__ void celu16(const uint32_t (&v)[16], const float (&b)[16], float sc, float alpha, float kexp, float (&x)[16]) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const f32x2 z = fma2(pack2(__uint_as_float(v[2 * i]), __uint_as_float(v[2 * i + 1])), pack2(sc, sc), pack2(b[2 * i], b[2 * i + 1]));
        float t0, t1, z0, z1, e0, e1;
        unpack2(mul2(z, pack2(kexp, kexp)), t0, t1);
        unpack2(fma2(pack2(fast_ex2(t0), fast_ex2(t1)), pack2(alpha, alpha), pack2(-alpha, -alpha)), e0, e1);
        unpack2(z, z0, z1);
        x[2 * i] = fmaxf(z0, fminf(e0, 0.f));
        x[2 * i + 1] = fmaxf(z1, fminf(e1, 0.f));
    }
}
// 16 accumulator columns -> (acc * sc) * CELU'(z) with CELU' recovered from the stored activation h (dcelu_from_h)
__device__ __forceinline__ void dcelu16(const uint32_t (&v)[16], const float (&h)[16], float sc, float inv_alpha, float (&x)[16]) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        float g0, g1;
        unpack2(fma2(pack2(h[2 * i], h[2 * i + 1]), pack2(inv_alpha, inv_alpha), pack2(1.0f, 1.0f)), g0, g1);
        const f32x2 a = mul2(pack2(__uint_as_float(v[2 * i]), __uint_as_float(v[2 * i + 1])), pack2(sc, sc));
        unpack2(mul2(a, pack2(fminf(g0, 1.0f), fminf(g1, 1.0f))), x[2 * i], x[2 * i + 1]);
    }
}
// tiled activation layout: element offset of (row tile rt, 64-column block kb) and, inside it, of (8-column group g, row r)
__device__ __forceinline__ size_t tile_off(int plane_tiles, int kblocks, int plane, int rt, int kb) {
    return ((size_t)(plane * plane_tiles + rt) * kblocks + kb) * (size_t)(BM * BK);
}
// 32 consecutive columns (4 groups) of one row -> hi and lo planes; tile pointers already include group and row
__device__ __forceinline__ void store_split32_tiled(const float (&x)[32], __half* hi_dst, __half* lo_dst) {
    uint32_t ph[16], pl[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) split_pair(x[2 * i], x[2 * i + 1], ph[i], pl[i]);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        *reinterpret_cast<uint4*>(hi_dst + i * (BM * 8)) = make_uint4(ph[4 * i], ph[4 * i + 1], ph[4 * i + 2], ph[4 * i + 3]);
        *reinterpret_cast<uint4*>(lo_dst + i * (BM * 8)) = make_uint4(pl[4 * i], pl[4 * i + 1], pl[4 * i + 2], pl[4 * i + 3]);
    }
}
__device__ __forceinline__ void load_joined32_tiled(const __half* hi_src, const __half* lo_src, float (&x)[32]) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const uint4 h = *reinterpret_cast<const uint4*>(hi_src + i * (BM * 8));
        const uint4 l = *reinterpret_cast<const uint4*>(lo_src + i * (BM * 8));
        unpack_add(h.x, l.x, x[8 * i + 0], x[8 * i + 1]);
        unpack_add(h.y, l.y, x[8 * i + 2], x[8 * i + 3]);
        unpack_add(h.z, l.z, x[8 * i + 4], x[8 * i + 5]);
        unpack_add(h.w, l.w, x[8 * i + 6], x[8 * i + 7]);
    }
}
__device__ __forceinline__ void load32(const float* __restrict__ src, float (&x)[32]) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const float4 v = __ldg(reinterpret_cast<const float4*>(src) + i);
        x[4 * i] = v.x; x[4 * i + 1] = v.y; x[4 * i + 2] = v.z; x[4 * i + 3] = v.w;
    }
}

// the (up to 4) feature blocks that column tile nt of a row tile produces: set bits 4 nt .. 4 nt + 3 of the mask
__device__ __forceinline__ int select_blocks(unsigned mask, int nt, int (&sel)[4]) {
    for (int i = 0; i < 4 * nt; ++i) mask &= mask - 1u;
    int n = 0;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        sel[i] = 0;
        if (mask) { sel[i] = __ffs(mask) - 1; mask &= mask - 1u; n = i + 1; }
    }
    return n;
}

template <int EPI, int CMP>
__global__ void __launch_bounds__(TC_THREADS, 1)
k_gemm_tc(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const TcArgs p) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;                      // SWIZZLE_128B tiles need 1024-byte alignment
    uint8_t* base_ptr = smem_raw + (base - raw);
    uint8_t* ostage_ptr = base_ptr + STAGES * STAGE_BYTES;                // output staging block of the CELU epilogue
    const uint32_t ostage = base + STAGES * STAGE_BYTES;
    uint64_t* bars = reinterpret_cast<uint64_t*>(base_ptr + STAGES * STAGE_BYTES + OUT_STAGE_BYTES);
    const uint32_t bar0 = base + STAGES * STAGE_BYTES + OUT_STAGE_BYTES;
    // barrier layout: full[STAGES], empty[STAGES], tfull[2], tempty[2], sfull[RING], sempty[RING], then the TMEM base
    // address word and the tile-id ring
    constexpr int NBARS = 2 * STAGES + 4 + 2 * RING;
    auto full_bar = [&](int s) { return bar0 + 8u * s; };
    auto empty_bar = [&](int s) { return bar0 + 8u * (STAGES + s); };
    auto tfull_bar = [&](int s) { return bar0 + 8u * (2 * STAGES + s); };
    auto tempty_bar = [&](int s) { return bar0 + 8u * (2 * STAGES + 2 + s); };
    auto sfull_bar = [&](int s) { return bar0 + 8u * (2 * STAGES + 4 + s); };
    auto sempty_bar = [&](int s) { return bar0 + 8u * (2 * STAGES + 4 + RING + s); };
    volatile uint32_t* tmem_word = reinterpret_cast<volatile uint32_t*>(bars + NBARS);
    volatile int* ring = reinterpret_cast<volatile int*>(bars + NBARS + 1);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_row_tiles = p.sp_start[NSP] / BM;
    const int ksplit = (EPI == EPI_GRAD && p.ksplit > 1) ? p.ksplit : 1;
    const int total_tiles = n_row_tiles * p.n_tiles * ksplit;
    const int KB = (p.K + BK - 1) / BK;
    const unsigned all_k = KB >= 32 ? 0xffffffffu : ((1u << KB) - 1u);
    // K blocks of split ks of a tile: [ks KB / ksplit, (ks + 1) KB / ksplit)
    auto split_mask = [&](int ks) -> unsigned {
        if (ksplit == 1) return 0xffffffffu;
        const int per = KB / ksplit;
        return ((per >= 32 ? 0xffffffffu : ((1u << per) - 1u)) << (ks * per));
    };

    if (warp == EPI_WARPS && lane == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
        for (int s = 0; s < 2; ++s) { mbar_init(tfull_bar(s), 1); mbar_init(tempty_bar(s), EPI_WARPS); }
        for (int s = 0; s < RING; ++s) { mbar_init(sfull_bar(s), 1); mbar_init(sempty_bar(s), 1 + EPI_WARPS); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        prefetch_tmap(&tmA);
        prefetch_tmap(&tmB);
    }
    if (warp == EPI_WARPS + 1) tmem_alloc(smem_u32((const void*)tmem_word), TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_word;

    // G1 visits only the K blocks that are non-zero for the row tile (an all-zero tile - isolated atoms - still
    // runs one block of zeros so that the accumulator is defined); everything else visits all of K.
    auto k_mask = [&](int rt) -> unsigned {
        if (CMP != CMP_K) return all_k;
        const unsigned m = p.tile_mask[rt];
        return m ? m : (1u << 14);
    };

    if (warp == EPI_WARPS) {
        // ===== tile scheduler + TMA producer =====
        if (elect_one()) {
            int stage = 0; uint32_t phase = 0;
            int slot = 0; uint32_t sphase = 0;
            for (;;) {
                int tile, rt = 0, nt = 0;
                for (;;) {
                    tile = atomicAdd(p.sched, 1);
                    if (tile >= total_tiles) { tile = -1; break; }
                    rt = (tile / ksplit) / p.n_tiles; nt = (tile / ksplit) - rt * p.n_tiles;
                    if (CMP != CMP_N || 4 * nt < __popc(p.tile_mask[rt])) break;      // B1: nothing to produce
                }
                mbar_wait(sempty_bar(slot), sphase ^ 1u);
                ring[slot] = tile;
                mbar_arrive(sfull_bar(slot));
                if (++slot == RING) { slot = 0; sphase ^= 1u; }
                if (tile < 0) break;
                const int row0 = rt * BM;
                const int s = max(p.row_species[row0], 0);
                int brow = (2 * s) * p.b_rows_per_species;
                int sel[4] = {0, 0, 0, 0};
                int nb = 0;
                uint32_t tx;
                if (CMP == CMP_N) {
                    nb = select_blocks(p.tile_mask[rt], nt, sel);
                    tx = 2u * A_PLANE_BYTES + 2u * (uint32_t)nb * NB_BLOCK_BYTES;
                } else {
                    brow += nt * p.b_rows_per_tile;
                    tx = 2u * A_PLANE_BYTES + 2u * (uint32_t)p.BN * BK * 2u;
                }
                for (unsigned km = k_mask(rt) & split_mask(tile % ksplit); km; km &= km - 1u) {
                    const int kb = __ffs(km) - 1;
                    mbar_wait(empty_bar(stage), phase ^ 1u);
                    const uint32_t sa = base + stage * STAGE_BYTES;
                    mbar_expect_tx(full_bar(stage), tx);
                    if (p.a_tiled) {
                        const int kba = p.a_kb_per_tile * nt + kb;
                        bulk_load(sa, p.a_tiled + tile_off(p.plane_tiles, p.a_kblocks, 0, rt, kba), A_PLANE_BYTES, full_bar(stage));
                        bulk_load(sa + A_PLANE_BYTES, p.a_tiled + tile_off(p.plane_tiles, p.a_kblocks, 1, rt, kba), A_PLANE_BYTES,
                                  full_bar(stage));
                    } else {
                        const int ka = p.a_k_off_per_tile * nt + kb * BK;
                        tma_load_2d(sa, &tmA, ka, row0, full_bar(stage));
                        tma_load_2d(sa + A_PLANE_BYTES, &tmA, ka, p.a_plane_rows + row0, full_bar(stage));
                    }
                    const uint32_t sb = sa + 2 * A_PLANE_BYTES;
                    if (CMP == CMP_N) {
#pragma unroll
                        for (int j = 0; j < 4; ++j)
                            if (j < nb) {
                                tma_load_2d(sb + j * NB_BLOCK_BYTES, &tmB, kb * BK, brow + sel[j] * KBLK, full_bar(stage));
                                tma_load_2d(sb + B_SLOT_BYTES + j * NB_BLOCK_BYTES, &tmB, kb * BK,
                                            brow + p.b_rows_per_species + sel[j] * KBLK, full_bar(stage));
                            }
                    } else {
                        tma_load_2d(sb, &tmB, kb * BK, brow, full_bar(stage));
                        tma_load_2d(sb + B_SLOT_BYTES, &tmB, kb * BK, brow + p.b_rows_per_species, full_bar(stage));
                    }
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else if (warp == EPI_WARPS + 1) {
        // ===== MMA issuer =====
        if (elect_one()) {
            int stage = 0; uint32_t phase = 0;
            int acc = 0; uint32_t acc_phase = 0;
            int slot = 0; uint32_t sphase = 0;
            for (;;) {
                mbar_wait(sfull_bar(slot), sphase);
                const int tile = ring[slot];
                mbar_arrive(sempty_bar(slot));
                if (++slot == RING) { slot = 0; sphase ^= 1u; }
                if (tile < 0) break;
                const int rt = (tile / ksplit) / p.n_tiles, nt = (tile / ksplit) - rt * p.n_tiles;
                int bn = p.BN;
                if (CMP == CMP_N) bn = KBLK * min(4, __popc(p.tile_mask[rt]) - 4 * nt);
                const uint32_t idesc = make_idesc(bn);
                mbar_wait(tempty_bar(acc), acc_phase ^ 1u);
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + (uint32_t)(acc * ACC_STRIDE);
                uint32_t accumulate = 0u;
                for (unsigned km = k_mask(rt) & split_mask(tile % ksplit); km; km &= km - 1u) {
                    const int kb = __ffs(km) - 1;
                    mbar_wait(full_bar(stage), phase);
                    tc_fence_after();
                    const uint32_t sa = base + stage * STAGE_BYTES;
                    const bool tiled = p.a_tiled != nullptr;
                    const uint64_t a_hi = tiled ? make_smem_desc_tiled(sa) : make_smem_desc(sa);
                    const uint64_t a_lo = tiled ? make_smem_desc_tiled(sa + A_PLANE_BYTES) : make_smem_desc(sa + A_PLANE_BYTES);
                    const uint64_t b_hi = make_smem_desc(sa + 2 * A_PLANE_BYTES);
                    const uint64_t b_lo = make_smem_desc(sa + 2 * A_PLANE_BYTES + B_SLOT_BYTES);
                    // one K step = 16 fp16: 32 bytes inside a swizzled 128-byte row, or two 8-column groups (4096 bytes) when tiled
                    const uint64_t a_step = tiled ? (uint64_t)(4096 >> 4) : 2u;
                    const int ksteps = min(BK / 16, (p.K - kb * BK) / 16);
                    for (int k = 0; k < ksteps; ++k) {
                        const uint64_t adv = (uint64_t)(k * 2), a_adv = (uint64_t)k * a_step;
                        umma_f16(d_tmem, a_hi + a_adv, b_hi + adv, idesc, accumulate);
                        if (!p.single) {
                            umma_f16(d_tmem, a_hi + a_adv, b_lo + adv, idesc, 1u);
                            umma_f16(d_tmem, a_lo + a_adv, b_hi + adv, idesc, 1u);
                        }
                        accumulate = 1u;
                    }
                    umma_commit(empty_bar(stage));                     // frees the smem stage when the MMAs retire
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
                umma_commit(tfull_bar(acc));                           // accumulator complete -> epilogue
                if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
            }
        }
    } else {
        // ===== epilogue (warps 0..7; a warp may touch only TMEM lanes 32*(warp%4) .. +31; the two warps of a
        //       lane quadrant take alternate 32-column chunks) =====
        const int q = warp & 3, half = warp >> 2;
        int acc = 0; uint32_t acc_phase = 0;
        int slot = 0; uint32_t sphase = 0;
        const float kexp = 1.4426950408889634f / p.alpha, inv_alpha = 1.0f / p.alpha;
        for (;;) {
            mbar_wait(sfull_bar(slot), sphase);
            const int tile = ring[slot];
            __syncwarp();
            if (lane == 0) mbar_arrive(sempty_bar(slot));
            if (++slot == RING) { slot = 0; sphase ^= 1u; }
            if (tile < 0) break;
            const int rt = (tile / ksplit) / p.n_tiles, nt = (tile / ksplit) - rt * p.n_tiles;
            const int row = rt * BM + q * 32 + lane;
            const int s = max(p.row_species[rt * BM], 0);
            const int ncols = p.n_tiles * p.BN;
            const int r_in = q * 32 + lane;
            int sel[4] = {0, 0, 0, 0};
            int bn = p.BN;
            if (CMP == CMP_N) bn = KBLK * select_blocks(p.tile_mask[rt], nt, sel);
            mbar_wait(tfull_bar(acc), acc_phase);
            tc_fence_after();
            const uint32_t t_row = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(acc * ACC_STRIDE);
            float e_acc = 0.f;
            for (int c0 = half * 32; c0 < bn; c0 += 64) {
                const int col = nt * p.BN + c0;
                uint32_t v[32];
                float x[32], aux[32];
                tmem_ld32_issue(t_row + (uint32_t)c0, v);
                if (EPI == EPI_CELU || EPI == EPI_OUT) load32(p.bias + (size_t)s * ncols + col, aux);
                // tiled output (and saved-activation) position of this thread's 32 columns
                const int ocol = nt * p.out_cols_per_tile + c0;
                const size_t in_tile = (size_t)(((ocol & 63) >> 3) * BM + r_in) * 8;
                const size_t o_hi = tile_off(p.plane_tiles, p.out_kblocks, 0, rt, ocol >> 6) + in_tile;
                const size_t o_lo = tile_off(p.plane_tiles, p.out_kblocks, 1, rt, ocol >> 6) + in_tile;
                if (EPI == EPI_DCELU) load_joined32_tiled(p.h_planes + o_hi, p.h_planes + o_lo, aux);
                tmem_ld_wait();
                if (EPI == EPI_CELU || EPI == EPI_OUT) {
#pragma unroll
                    for (int i = 0; i < 32; ++i) x[i] = celu_f(fmaf(__uint_as_float(v[i]), p.acc_scale, aux[i]), p.alpha, kexp);
                }
                if (EPI == EPI_CELU) {
                    // The 64-column block (all 8 epilogue warps, 32 KB as hi plane + lo plane) is assembled in shared memory in
                    // its global (tiled) layout and leaves as two bulk copies.  BN is a multiple of 64 here, so every warp runs
                    // the same number of rounds and the two named barriers per round are uniform.
                    if (warp == 0 && lane == 0) bulk_wait_read<0>();        // the previous block's copies have read the buffer
                    named_bar(1, 32 * EPI_WARPS);
                    {
                        uint8_t* dst = ostage_ptr + (size_t)(((ocol & 63) >> 3) * BM + r_in) * 16;
                        uint32_t ph[16], pl[16];
#pragma unroll
                        for (int i = 0; i < 16; ++i) split_pair(x[2 * i], x[2 * i + 1], ph[i], pl[i]);
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            *reinterpret_cast<uint4*>(dst + i * (BM * 16)) = make_uint4(ph[4 * i], ph[4 * i + 1], ph[4 * i + 2], ph[4 * i + 3]);
                            *reinterpret_cast<uint4*>(dst + A_PLANE_BYTES + i * (BM * 16)) = make_uint4(pl[4 * i], pl[4 * i + 1], pl[4 * i + 2], pl[4 * i + 3]);
                        }
                    }
                    fence_async_smem();
                    named_bar(1, 32 * EPI_WARPS);
                    if (warp == 0 && lane == 0) {
                        bulk_store(p.out_planes + tile_off(p.plane_tiles, p.out_kblocks, 0, rt, ocol >> 6), ostage, A_PLANE_BYTES);
                        bulk_store(p.out_planes + tile_off(p.plane_tiles, p.out_kblocks, 1, rt, ocol >> 6), ostage + A_PLANE_BYTES, A_PLANE_BYTES);
                        bulk_commit();
                    }
                } else if (EPI == EPI_OUT) {
                    load32(p.w4 + (size_t)s * ncols + col, aux);
                    const float dsc = p.inv_models * D_SCALE;
#pragma unroll
                    for (int i = 0; i < 32; ++i) {
                        e_acc = fmaf(aux[i], x[i], e_acc);
                        x[i] = aux[i] * dsc * dcelu_from_h(x[i], inv_alpha);
                    }
                    store_split32_tiled(x, p.out_planes + o_hi, p.out_planes + o_lo);
                } else if (EPI == EPI_DCELU) {
#pragma unroll
                    for (int i = 0; i < 32; ++i) x[i] = __uint_as_float(v[i]) * p.acc_scale * dcelu_from_h(aux[i], inv_alpha);
                    store_split32_tiled(x, p.out_planes + o_hi, p.out_planes + o_lo);
                } else {   // EPI_GRAD
                    int gcol = col;
                    if (CMP == CMP_N) {                                  // chunk c0 belongs to the (c0/64)-th selected block
                        const int j = c0 >> 6;
                        const int blk = j == 0 ? sel[0] : j == 1 ? sel[1] : j == 2 ? sel[2] : sel[3];
                        gcol = blk * KBLK + (c0 & 63);
                    }
                    float4* dst = reinterpret_cast<float4*>(p.out_f32 + (size_t)row * p.out_ld + gcol);
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const float4 o = make_float4(__uint_as_float(v[4 * i]) * p.acc_scale, __uint_as_float(v[4 * i + 1]) * p.acc_scale,
                                                     __uint_as_float(v[4 * i + 2]) * p.acc_scale, __uint_as_float(v[4 * i + 3]) * p.acc_scale);
                        if (ksplit == 1) dst[i] = o;
                        else atomicAdd(dst + i, o);              // partial sum over this item's K blocks (16-byte vector atomic)
                    }
                }
            }
            if (EPI == EPI_OUT) atomicAdd(&p.e_atom[row], (e_acc + (half == 0 ? p.b4[s * p.n_tiles + nt] : 0.f)) * p.inv_models);
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tempty_bar(acc));
            if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
        }
        if (EPI == EPI_CELU && warp == 0 && lane == 0) bulk_wait_all();    // the last block's copies are complete before the CTA exits
    }
    tc_fence_before();
    __syncthreads();
    if (warp == EPI_WARPS + 1) tmem_dealloc(tmem_base, TMEM_COLS);
}

// ======================================================================================================
// G1 and B1 with TWO row tiles per CTA.  Experiments (profiles/r2b_*.md) show the one-tile kernel above bound by the
// chip-wide L2 -> SM throughput (about 50 B/clk/SM with all 148 SMs streaming): one 64-wide K block of one 128-row tile
// brings 96 KB (A 32 KB, W 64 KB) for 1 536 MMA cycles.  Here the two row tiles of a pair (same species, same feature-
// block mask: nlist.cu keeps both pair-uniform) share every weight K block: W is fetched once, the MMAs of tile 0
// accumulate into TMEM columns [0, 256) and those of tile 1 into [256, 512).  Per K block: 128 KB for 3 072 MMA cycles
// (42 B/clk) in G1, and for a 3-block column tile of B1 112 KB for 2 304 cycles (49 B/clk, was 71).  The price: both
// accumulator stages belong to the item in flight, so the epilogue of an item overlaps only the first K blocks of the
// next one (tile 0's accumulator is released first) - small against B1's 32 K blocks, visible in G1.
//   smem: W ring 2 x 64 KB (hi plane, lo plane), A ring 3 x 32 KB (hi, lo); roles as in k_gemm_tc.
// ======================================================================================================
constexpr int T2_WSLOTS = 2, T2_ASLOTS = 3;
constexpr int T2_W_BYTES = 2 * B_SLOT_BYTES;          // 64 KB
constexpr int T2_A_BYTES = 2 * A_PLANE_BYTES;         // 32 KB
constexpr int T2_SMEM = T2_WSLOTS * T2_W_BYTES + T2_ASLOTS * T2_A_BYTES + 1024 /*align*/ + 256 /*barriers, TMEM word, ring*/;

template <int EPI, int CMP>
__global__ void __launch_bounds__(TC_THREADS, 1)
k_gemm_tc2(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const TcArgs p) {
    static_assert((EPI == EPI_CELU && CMP == CMP_K) || (EPI == EPI_GRAD && CMP == CMP_N), "two-tile kernel: G1 and B1 only");
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;
    uint8_t* base_ptr = smem_raw + (base - raw);
    const uint32_t wring = base, aring = base + T2_WSLOTS * T2_W_BYTES;
    constexpr int DATA = T2_WSLOTS * T2_W_BYTES + T2_ASLOTS * T2_A_BYTES;
    uint64_t* bars = reinterpret_cast<uint64_t*>(base_ptr + DATA);
    const uint32_t bar0 = base + DATA;
    // barriers: wfull[2], wempty[2], afull[3], aempty[3], tfull[2], tempty[2], sfull[RING], sempty[RING]
    constexpr int NBARS = 2 * T2_WSLOTS + 2 * T2_ASLOTS + 4 + 2 * RING;
    auto wfull_bar = [&](int s) { return bar0 + 8u * s; };
    auto wempty_bar = [&](int s) { return bar0 + 8u * (T2_WSLOTS + s); };
    auto afull_bar = [&](int s) { return bar0 + 8u * (2 * T2_WSLOTS + s); };
    auto aempty_bar = [&](int s) { return bar0 + 8u * (2 * T2_WSLOTS + T2_ASLOTS + s); };
    auto tfull_bar = [&](int s) { return bar0 + 8u * (2 * T2_WSLOTS + 2 * T2_ASLOTS + s); };
    auto tempty_bar = [&](int s) { return bar0 + 8u * (2 * T2_WSLOTS + 2 * T2_ASLOTS + 2 + s); };
    auto sfull_bar = [&](int s) { return bar0 + 8u * (2 * T2_WSLOTS + 2 * T2_ASLOTS + 4 + s); };
    auto sempty_bar = [&](int s) { return bar0 + 8u * (2 * T2_WSLOTS + 2 * T2_ASLOTS + 4 + RING + s); };
    volatile uint32_t* tmem_word = reinterpret_cast<volatile uint32_t*>(bars + NBARS);
    volatile int* ring = reinterpret_cast<volatile int*>(bars + NBARS + 1);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_pairs = p.sp_start[NSP] / (2 * BM);            // species groups are aligned to 256 rows
    const int total_items = n_pairs * p.n_tiles;
    const int KB = (p.K + BK - 1) / BK;
    const unsigned all_k = KB >= 32 ? 0xffffffffu : ((1u << KB) - 1u);

    if (warp == EPI_WARPS && lane == 0) {
        for (int s = 0; s < T2_WSLOTS; ++s) { mbar_init(wfull_bar(s), 1); mbar_init(wempty_bar(s), 1); }
        for (int s = 0; s < T2_ASLOTS; ++s) { mbar_init(afull_bar(s), 1); mbar_init(aempty_bar(s), 1); }
        for (int s = 0; s < 2; ++s) { mbar_init(tfull_bar(s), 1); mbar_init(tempty_bar(s), EPI_WARPS); }
        for (int s = 0; s < RING; ++s) { mbar_init(sfull_bar(s), 1); mbar_init(sempty_bar(s), 1 + EPI_WARPS); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        prefetch_tmap(&tmA);
        prefetch_tmap(&tmB);
    }
    if (warp == EPI_WARPS + 1) tmem_alloc(smem_u32((const void*)tmem_word), TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_word;

    // tile masks are pair-uniform (nlist.cu): the first tile's mask speaks for both
    auto k_mask = [&](int pr) -> unsigned {
        if (CMP != CMP_K) return all_k;
        const unsigned m = p.tile_mask[2 * pr];
        return m ? m : (1u << 14);                             // an all-zero pair still runs one block of zeros
    };

    if (warp == EPI_WARPS) {
        // ===== item scheduler + producer =====
        if (elect_one()) {
            int ws = 0; uint32_t wphase = 0;
            int as = 0; uint32_t aphase = 0;
            int slot = 0; uint32_t sphase = 0;
            for (;;) {
                int item, pr = 0, nt = 0;
                for (;;) {
                    int t = atomicAdd(p.sched, 1);
                    if (CMP == CMP_N) {
                        // B1: an item's cost is its number of feature blocks (1..4) x all of K, and there are only a few
                        // items per SM: hand them out LONGEST FIRST (four passes over the items: 4, 3, 2, 1 blocks), so that
                        // the tail of the launch is made of short items
                        if (t >= 4 * total_items) { item = -1; break; }
                        const int pass = t / total_items;
                        item = t - pass * total_items;
                        pr = item / p.n_tiles; nt = item - pr * p.n_tiles;
                        if (min(4, __popc(p.tile_mask[2 * pr]) - 4 * nt) == 4 - pass) break;
                    } else {
                        item = t;
                        if (item >= total_items) { item = -1; break; }
                        pr = item / p.n_tiles; nt = item - pr * p.n_tiles;
                        break;
                    }
                }
                mbar_wait(sempty_bar(slot), sphase ^ 1u);
                ring[slot] = item;
                mbar_arrive(sfull_bar(slot));
                if (++slot == RING) { slot = 0; sphase ^= 1u; }
                if (item < 0) break;
                const int s = max(p.row_species[2 * pr * BM], 0);
                int brow = (2 * s) * p.b_rows_per_species;
                int sel[4] = {0, 0, 0, 0};
                int nb = 0;
                uint32_t wtx;
                if (CMP == CMP_N) {
                    nb = select_blocks(p.tile_mask[2 * pr], nt, sel);
                    wtx = 2u * (uint32_t)nb * NB_BLOCK_BYTES;
                } else {
                    brow += nt * p.b_rows_per_tile;
                    wtx = 2u * (uint32_t)p.BN * BK * 2u;
                }
                for (unsigned km = k_mask(pr); km; km &= km - 1u) {
                    const int kb = __ffs(km) - 1;
                    // the weight K block, once for both row tiles
                    mbar_wait(wempty_bar(ws), wphase ^ 1u);
                    const uint32_t sb = wring + ws * T2_W_BYTES;
                    mbar_expect_tx(wfull_bar(ws), wtx);
                    if (CMP == CMP_N) {
#pragma unroll
                        for (int j = 0; j < 4; ++j)
                            if (j < nb) {
                                tma_load_2d(sb + j * NB_BLOCK_BYTES, &tmB, kb * BK, brow + sel[j] * KBLK, wfull_bar(ws));
                                tma_load_2d(sb + B_SLOT_BYTES + j * NB_BLOCK_BYTES, &tmB, kb * BK,
                                            brow + p.b_rows_per_species + sel[j] * KBLK, wfull_bar(ws));
                            }
                    } else {
                        tma_load_2d(sb, &tmB, kb * BK, brow, wfull_bar(ws));
                        tma_load_2d(sb + B_SLOT_BYTES, &tmB, kb * BK, brow + p.b_rows_per_species, wfull_bar(ws));
                    }
                    if (++ws == T2_WSLOTS) { ws = 0; wphase ^= 1u; }
                    // the A tiles of the two rows tiles
#pragma unroll
                    for (int r = 0; r < 2; ++r) {
                        const int rt = 2 * pr + r;
                        mbar_wait(aempty_bar(as), aphase ^ 1u);
                        const uint32_t sa = aring + as * T2_A_BYTES;
                        mbar_expect_tx(afull_bar(as), (uint32_t)T2_A_BYTES);
                        if (p.a_tiled) {
                            const int kba = p.a_kb_per_tile * nt + kb;
                            bulk_load(sa, p.a_tiled + tile_off(p.plane_tiles, p.a_kblocks, 0, rt, kba), A_PLANE_BYTES, afull_bar(as));
                            bulk_load(sa + A_PLANE_BYTES, p.a_tiled + tile_off(p.plane_tiles, p.a_kblocks, 1, rt, kba), A_PLANE_BYTES,
                                      afull_bar(as));
                        } else {
                            const int ka = p.a_k_off_per_tile * nt + kb * BK;
                            tma_load_2d(sa, &tmA, ka, rt * BM, afull_bar(as));
                            tma_load_2d(sa + A_PLANE_BYTES, &tmA, ka, p.a_plane_rows + rt * BM, afull_bar(as));
                        }
                        if (++as == T2_ASLOTS) { as = 0; aphase ^= 1u; }
                    }
                }
            }
        }
    } else if (warp == EPI_WARPS + 1) {
        // ===== MMA issuer =====
        if (elect_one()) {
            int ws = 0; uint32_t wphase = 0;
            int as = 0; uint32_t aphase = 0;
            uint32_t acc_phase = 0;
            int slot = 0; uint32_t sphase = 0;
            for (;;) {
                mbar_wait(sfull_bar(slot), sphase);
                const int item = ring[slot];
                mbar_arrive(sempty_bar(slot));
                if (++slot == RING) { slot = 0; sphase ^= 1u; }
                if (item < 0) break;
                const int pr = item / p.n_tiles, nt = item - pr * p.n_tiles;
                int bn = p.BN;
                if (CMP == CMP_N) bn = KBLK * min(4, __popc(p.tile_mask[2 * pr]) - 4 * nt);
                const uint32_t idesc = make_idesc(bn);
                uint32_t accumulate = 0u;
                const bool tiled = p.a_tiled != nullptr;
                const uint64_t a_step = tiled ? (uint64_t)(4096 >> 4) : 2u;
                for (unsigned km = k_mask(pr); km; km &= km - 1u) {
                    const int kb = __ffs(km) - 1;
                    mbar_wait(wfull_bar(ws), wphase);
                    const uint32_t sb = wring + ws * T2_W_BYTES;
                    const uint64_t b_hi = make_smem_desc(sb), b_lo = make_smem_desc(sb + B_SLOT_BYTES);
                    const int ksteps = min(BK / 16, (p.K - kb * BK) / 16);
#pragma unroll
                    for (int r = 0; r < 2; ++r) {
                        if (accumulate == 0u) {                       // first K block of the item: the accumulator must be drained
                            mbar_wait(tempty_bar(r), acc_phase ^ 1u);
                        }
                        mbar_wait(afull_bar(as), aphase);
                        tc_fence_after();
                        const uint32_t sa = aring + as * T2_A_BYTES;
                        const uint64_t a_hi = tiled ? make_smem_desc_tiled(sa) : make_smem_desc(sa);
                        const uint64_t a_lo = tiled ? make_smem_desc_tiled(sa + A_PLANE_BYTES) : make_smem_desc(sa + A_PLANE_BYTES);
                        const uint32_t d_tmem = tmem_base + (uint32_t)(r * ACC_STRIDE);
                        for (int k = 0; k < ksteps; ++k) {
                            const uint64_t adv = (uint64_t)(k * 2), a_adv = (uint64_t)k * a_step;
                            umma_f16(d_tmem, a_hi + a_adv, b_hi + adv, idesc, (accumulate | (uint32_t)(k > 0)));
                            if (!p.single) {
                                umma_f16(d_tmem, a_hi + a_adv, b_lo + adv, idesc, 1u);
                                umma_f16(d_tmem, a_lo + a_adv, b_hi + adv, idesc, 1u);
                            }
                        }
                        umma_commit(aempty_bar(as));
                        if (++as == T2_ASLOTS) { as = 0; aphase ^= 1u; }
                    }
                    accumulate = 1u;
                    umma_commit(wempty_bar(ws));
                    if (++ws == T2_WSLOTS) { ws = 0; wphase ^= 1u; }
                }
                umma_commit(tfull_bar(0));                             // both accumulators complete -> epilogue
                umma_commit(tfull_bar(1));
                acc_phase ^= 1u;
            }
        }
    } else {
        // ===== epilogue (warps 0..7): tile 0's accumulator first, so that the next item's MMAs can start on it =====
        const int q = warp & 3, half = warp >> 2;
        uint32_t acc_phase = 0;
        int slot = 0; uint32_t sphase = 0;
        const float kexp = 1.4426950408889634f / p.alpha;
        for (;;) {
            mbar_wait(sfull_bar(slot), sphase);
            const int item = ring[slot];
            __syncwarp();
            if (lane == 0) mbar_arrive(sempty_bar(slot));
            if (++slot == RING) { slot = 0; sphase ^= 1u; }
            if (item < 0) break;
            const int pr = item / p.n_tiles, nt = item - pr * p.n_tiles;
            const int s = max(p.row_species[2 * pr * BM], 0);
            const int ncols = p.n_tiles * p.BN;
            const int r_in = q * 32 + lane;
            int sel[4] = {0, 0, 0, 0};
            int bn = p.BN;
            if (CMP == CMP_N) bn = KBLK * select_blocks(p.tile_mask[2 * pr], nt, sel);
#pragma unroll 1
            for (int r = 0; r < 2; ++r) {
                const int rt = 2 * pr + r;
                const int row = rt * BM + r_in;
                mbar_wait(tfull_bar(r), acc_phase);
                tc_fence_after();
                const uint32_t t_row = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(r * ACC_STRIDE);
                for (int c0 = half * 32; c0 < bn; c0 += 64) {
                    const int col = nt * p.BN + c0;
                    uint32_t v[32];
                    tmem_ld32_issue(t_row + (uint32_t)c0, v);
                    if (EPI == EPI_CELU) {
                        float x[32], aux[32];
                        load32(p.bias + (size_t)s * ncols + col, aux);
                        const int ocol = nt * p.out_cols_per_tile + c0;
                        const size_t in_tile = (size_t)(((ocol & 63) >> 3) * BM + r_in) * 8;
                        const size_t o_hi = tile_off(p.plane_tiles, p.out_kblocks, 0, rt, ocol >> 6) + in_tile;
                        const size_t o_lo = tile_off(p.plane_tiles, p.out_kblocks, 1, rt, ocol >> 6) + in_tile;
                        tmem_ld_wait();
#pragma unroll
                        for (int i = 0; i < 32; ++i) x[i] = celu_f(fmaf(__uint_as_float(v[i]), p.acc_scale, aux[i]), p.alpha, kexp);
                        store_split32_tiled(x, p.out_planes + o_hi, p.out_planes + o_lo);
                    } else {   // EPI_GRAD: chunk c0 belongs to the (c0/64)-th selected block
                        const int j = c0 >> 6;
                        const int blk = j == 0 ? sel[0] : j == 1 ? sel[1] : j == 2 ? sel[2] : sel[3];
                        const int gcol = blk * KBLK + (c0 & 63);
                        float4* dst = reinterpret_cast<float4*>(p.out_f32 + (size_t)row * p.out_ld + gcol);
                        tmem_ld_wait();
#pragma unroll
                        for (int i = 0; i < 8; ++i)
                            dst[i] = make_float4(__uint_as_float(v[4 * i]) * p.acc_scale, __uint_as_float(v[4 * i + 1]) * p.acc_scale,
                                                 __uint_as_float(v[4 * i + 2]) * p.acc_scale, __uint_as_float(v[4 * i + 3]) * p.acc_scale);
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(tempty_bar(r));
            }
            acc_phase ^= 1u;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == EPI_WARPS + 1) tmem_dealloc(tmem_base, TMEM_COLS);
#ifdef T2_TRACE
    if (EPI == EPI_GRAD && threadIdx.x == 0) { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); printf("T2END %d %llu\n", (int)blockIdx.x, t); }
#endif
}

// ======================================================================================================
// (A cta_group::2 variant of G1 / B1 - k_gemm_pair: two row tiles per MMA, half of the weight tile per CTA, cost-balanced
// static schedule - lived here in rounds 1-2.  Measured twice, never faster than k_gemm_tc2: removed in round 3; the
// measurements are in DESIGN.md §6.3.)

// ======================================================================================================
// Fused middle of the chain.  G2, G3, B3 and B2 are small GEMMs whose split-fp16 activations (4 B per element)
// cost more HBM time than MMA time when every layer is its own launch (profiles/r1c: 66-81 % DRAM).  Here one
// work item = (row tile, network) runs   h1 -> h2 -> (E_i, d3) -> d2 -> d1   inside one CTA, and the four GEMMs and
// their epilogues are software-pipelined at 64-column granularity: the epilogue of GEMM p produces the A operand of
// GEMM p+1 in 64-column blocks (= K blocks of p+1) and signals each block, so the MMAs of p+1 start after the first
// epilogue round and run under the remaining ones.
//   * h2 and d2 live in ONE 96 KB shared-memory region X as the no-swizzle K-major A operand (d2 overwrites h2 in
//     place: B3's epilogue thread reads h2(r, n) for CELU'(z2) and writes d2(r, n) to the same bytes);
//   * d3 is the A operand of B3 straight from TENSOR MEMORY (tcgen05.mma with A in TMEM: lane = row, 16-bit
//     elements packed two per column along K), written by G3's epilogue with tcgen05.st - so h2 stays intact in X
//     until B3's epilogue has used it and no activation needs a second shared-memory region;
//   * weights stream from L2 as pre-tiled images (the exact shared-memory image of one 16-wide K step of one GEMM,
//     hi plane then lo plane, fetched by one plain cp.async.bulk; no tensor map) through a ring of 6 x 20 KB slots;
//     h1 (tiled activation layout) streams through the same slots.
// TMEM (512 columns, all used): P = [0,192) accumulator of G2 and of B3; Q = [192,352) accumulator of G3;
// D = [352,512) d3 as fp16 A operand (hi 80 columns, lo 80 columns); B2 accumulates into Q u D = [192,448).
// Every reuse is ordered by the data dependencies themselves (see the hazard notes at the barriers).
// ======================================================================================================
#ifndef MID_DBG
#define MID_DBG 0      // timing experiments only: 1 = epilogues without work, 2 = no MMAs issued, 4 = no d1 stores, 8 = half the weight bytes
#endif
#define MID_WB(x) ((MID_DBG & 8) ? (x) / 2u : (x))
#ifndef FU_BULK_H1
#define FU_BULK_H1 0   // k_mlp_fused: h1 blocks 0..2 reach the scratch tile as bulk copies out of X (1) or as plain stores of the epilogue threads (0)
#endif
#ifndef FU_BULK_D1
#define FU_BULK_D1 1   // k_mlp_fused: d1 blocks 0..2 are written over h1 in X and leave as bulk copies (1), or plain stores (0)
#endif
#ifndef MID_TRACE
#define MID_TRACE 0    // timing experiments only: CTA 0 records clock64() per role for a few items and prints them at the end
#endif
#if MID_TRACE
__device__ long long g_tr[3][8][24];
#define TR(role, it, ev) do { if (blockIdx.x == 0 && (it) >= 8 && (it) < 16) g_tr[role][(it) - 8][ev] = clock64(); } while (0)
#else
#define TR(role, it, ev) do { } while (0)
#endif
constexpr int MID_SLOTS = 3;                     // ring slots of TWO 16-wide K steps each: one full-barrier wait and one commit per 6 MMAs
constexpr int MID_SLOT_BYTES = 40960;
constexpr int MID_A_OFF = 24576;                 // G2 slots: W2 images of the two K steps (24 KB), then h1 hi (8 KB), h1 lo (8 KB)
constexpr int MID_X_PLANE = BM * H2 * 2;         // 48 KB per plane
constexpr int MID_X_BYTES = 2 * MID_X_PLANE;
constexpr int MID_CONST_FLOATS = H2 + H3 + H3;   // b2, b3, w4 of one (species, network), staged in shared memory (two buffers)
constexpr int MID_CONST_BYTES = MID_CONST_FLOATS * 4;
constexpr int MID_H_ROUND = 32768;               // one 64-column block of h1, hi plane then lo plane (B2's epilogue reads it from X)
constexpr int MID_SMEM = MID_X_BYTES + MID_SLOTS * MID_SLOT_BYTES + 2 * MID_CONST_BYTES + 1024 /*align*/ + 512 /*barriers, TMEM word, ring*/;
static_assert(3 * MID_H_ROUND == MID_X_BYTES, "three rounds of h1 fill X exactly");
constexpr uint32_t MID_P = 0, MID_Q = 192, MID_D = 352, MID_D_LO = MID_D + H3 / 2;
static_assert(MID_D_LO + H3 / 2 == TMEM_COLS && MID_Q + H1 <= TMEM_COLS, "TMEM map");
// weight image of one (species, network), in halves: per GEMM [K step][plane][8-column group (2)][n][8]
constexpr int MID_W_G2 = 0;
constexpr int MID_W_G3 = MID_W_G2 + (H1 / 16) * 32 * H2;
constexpr int MID_W_B3 = MID_W_G3 + (H2 / 16) * 32 * H3;
constexpr int MID_W_B2 = MID_W_B3 + (H3 / 16) * 32 * H2;
constexpr int MID_W_TOTAL = MID_W_B2 + (H2 / 16) * 32 * H1;

constexpr int MID_EPI_WARPS = 16;    // four per TMEM lane quadrant, each taking every fourth 16-column chunk
constexpr int MID_THREADS = 64 + 32 * MID_EPI_WARPS;

__device__ __forceinline__ void tmem_ld16_issue(uint32_t taddr, uint32_t (&v)[16]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t (&v)[8]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};"
                 ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7])
                 : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// D[tmem] (+)= A[tmem] * B[smem]: A is M x 16 fp16 in tensor memory (lane = row, two K elements per column)
__device__ __forceinline__ void umma_f16_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
        ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void load16(const float* __restrict__ src, float (&x)[16]) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float4 v = __ldg(reinterpret_cast<const float4*>(src) + i);
        x[4 * i] = v.x; x[4 * i + 1] = v.y; x[4 * i + 2] = v.z; x[4 * i + 3] = v.w;
    }
}

struct MidArgs {
    int single;               // 1: single-pass fp16 (hi x hi only)
    const int* row_species;
    const int* sp_start;
    int n_models;
    int plane_tiles;          // row tiles per plane of the activation buffers
    const __half* h1;         // tiled activation planes, n_models*4 64-column blocks per row tile
    __half* d1;               // same geometry
    const __half* wimg;       // [species][network][MID_W_TOTAL]
    const float *b2, *b3, *w4, *b4;
    float inv_models, alpha;
    float* e_atom;
    int* sched;
    int forward_only;         // stop after G3's epilogue (energies only): no d3, B3, B2, d1
};

// K-major operand without swizzle, [8-column group][row][16 B]: leading byte offset = next group (rows * 16), stride
// byte offset (next 8 rows) 128
__device__ __forceinline__ uint64_t make_desc_ns(uint32_t saddr, uint32_t lbo_bytes) {
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFF) >> 4);
    d |= (uint64_t)(lbo_bytes >> 4) << 16;
    d |= (uint64_t)(128 >> 4) << 32;
    d |= (uint64_t)1 << 46;
    return d;
}

// 16 consecutive columns c0.. of row r -> hi / lo planes of X
__device__ __forceinline__ void store_split16_x(const float (&x)[16], uint8_t* xp, int c0, int r_in) {
    uint32_t ph[8], pl[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) split_pair(x[2 * i], x[2 * i + 1], ph[i], pl[i]);
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        uint8_t* dst = xp + (size_t)(((c0 >> 3) + i) * BM + r_in) * 16;
        *reinterpret_cast<uint4*>(dst) = make_uint4(ph[4 * i], ph[4 * i + 1], ph[4 * i + 2], ph[4 * i + 3]);
        *reinterpret_cast<uint4*>(dst + MID_X_PLANE) = make_uint4(pl[4 * i], pl[4 * i + 1], pl[4 * i + 2], pl[4 * i + 3]);
    }
}
// the same to the tiled activation planes in global memory (pointers include group and row)
__device__ __forceinline__ void store_split16_tiled(const float (&x)[16], __half* hi_dst, __half* lo_dst) {
    uint32_t ph[8], pl[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) split_pair(x[2 * i], x[2 * i + 1], ph[i], pl[i]);
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        *reinterpret_cast<uint4*>(hi_dst + i * (BM * 8)) = make_uint4(ph[4 * i], ph[4 * i + 1], ph[4 * i + 2], ph[4 * i + 3]);
        *reinterpret_cast<uint4*>(lo_dst + i * (BM * 8)) = make_uint4(pl[4 * i], pl[4 * i + 1], pl[4 * i + 2], pl[4 * i + 3]);
    }
}
__device__ __forceinline__ void join16(const uint4 (&h)[2], const uint4 (&l)[2], float (&x)[16]) {
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        unpack_add(h[i].x, l[i].x, x[8 * i + 0], x[8 * i + 1]);
        unpack_add(h[i].y, l[i].y, x[8 * i + 2], x[8 * i + 3]);
        unpack_add(h[i].z, l[i].z, x[8 * i + 4], x[8 * i + 5]);
        unpack_add(h[i].w, l[i].w, x[8 * i + 6], x[8 * i + 7]);
    }
}

__global__ void __launch_bounds__(MID_THREADS, 1)
k_mlp_mid(const MidArgs p) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;
    uint8_t* x_ptr = smem_raw + (base - raw);                         // X region (generic pointer), xs its shared address
    const uint32_t xs = base;
    const uint32_t slots = base + MID_X_BYTES;
    const uint32_t cst_s = slots + MID_SLOTS * MID_SLOT_BYTES;        // per-item constants b2 | b3 | w4, two buffers
    const float* cst_ptr = reinterpret_cast<const float*>(x_ptr + MID_X_BYTES + MID_SLOTS * MID_SLOT_BYTES);
    const uint32_t bar0 = cst_s + 2 * MID_CONST_BYTES;
    uint64_t* bars = reinterpret_cast<uint64_t*>(x_ptr + MID_X_BYTES + MID_SLOTS * MID_SLOT_BYTES + 2 * MID_CONST_BYTES);
    // barriers: full[SLOTS], empty[SLOTS], acc_p, acc_q, xr[3], xfree, hfull[3], cfull[2], cempty[2], sfull[RING], sempty[RING];
    // then the TMEM word and the item ring
    constexpr int NBARS = 2 * MID_SLOTS + 13 + 2 * RING;
    auto full_bar = [&](int s) { return bar0 + 8u * s; };
    auto empty_bar = [&](int s) { return bar0 + 8u * (MID_SLOTS + s); };
    const uint32_t accp_bar = bar0 + 8u * (2 * MID_SLOTS), accq_bar = accp_bar + 8u;
    auto xr_bar = [&](int k) { return accp_bar + 16u + 8u * k; };      // 64-column block k of an epilogue's output is ready
    const uint32_t xfree_bar = accp_bar + 40u;                         // B2's MMAs have completed: X (d2) is dead
    auto hfull_bar = [&](int k) { return accp_bar + 48u + 8u * k; };   // h1 block k of the item has landed in X (for CELU'(z1))
    auto cfull_bar = [&](int b) { return accp_bar + 72u + 8u * b; };
    auto cempty_bar = [&](int b) { return accp_bar + 88u + 8u * b; };
    auto sfull_bar = [&](int s) { return bar0 + 8u * (2 * MID_SLOTS + 13 + s); };
    auto sempty_bar = [&](int s) { return bar0 + 8u * (2 * MID_SLOTS + 13 + RING + s); };
    volatile uint32_t* tmem_word = reinterpret_cast<volatile uint32_t*>(bars + NBARS);
    volatile int* ring = reinterpret_cast<volatile int*>(bars + NBARS + 1);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int M = p.n_models;
    const int total_items = (p.sp_start[NSP] / BM) * M;

    if (warp == MID_EPI_WARPS && lane == 0) {
        for (int s = 0; s < MID_SLOTS; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
        mbar_init(accp_bar, 1); mbar_init(accq_bar, 1); mbar_init(xfree_bar, 1);
        for (int k = 0; k < 3; ++k) { mbar_init(xr_bar(k), MID_EPI_WARPS); mbar_init(hfull_bar(k), 1); }
        for (int b = 0; b < 2; ++b) { mbar_init(cfull_bar(b), 1); mbar_init(cempty_bar(b), MID_EPI_WARPS); }
        for (int s = 0; s < RING; ++s) { mbar_init(sfull_bar(s), 1); mbar_init(sempty_bar(s), 1 + MID_EPI_WARPS); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == MID_EPI_WARPS + 1) tmem_alloc(smem_u32((const void*)tmem_word), TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_word;

    if (warp == MID_EPI_WARPS) {
        // ===== item scheduler + producer =====
        if (elect_one()) {
            int slot = 0; uint32_t phase = 0;
            int rs = 0; uint32_t rphase = 0;
            int cb = 0; uint32_t cphase = 0;
            uint32_t hphase = 0;
            int prev_rt = -1, prev_e = 0;
            auto next_slot = [&]() -> uint32_t {
                mbar_wait(empty_bar(slot), phase ^ 1u);
                return slots + (uint32_t)slot * MID_SLOT_BYTES;
            };
            auto advance = [&]() { if (++slot == MID_SLOTS) { slot = 0; phase ^= 1u; } };
            // h1 of the PREVIOUS item -> X once its B2 MMAs (the last readers of d2 in X) have completed: three 64-column
            // blocks (hi plane then lo plane) for CELU'(z1) in B2's epilogue; the fourth block comes by plain loads
            auto load_h1_for_b2 = [&]() {
                mbar_wait(xfree_bar, hphase); hphase ^= 1u;
                for (int k = 0; k < 3; ++k) {
                    mbar_expect_tx(hfull_bar(k), (uint32_t)MID_H_ROUND);
                    bulk_load(xs + (uint32_t)(k * MID_H_ROUND), p.h1 + tile_off(p.plane_tiles, M * 4, 0, prev_rt, prev_e * 4 + k), 16384u, hfull_bar(k));
                    bulk_load(xs + (uint32_t)(k * MID_H_ROUND) + 16384u, p.h1 + tile_off(p.plane_tiles, M * 4, 1, prev_rt, prev_e * 4 + k), 16384u,
                              hfull_bar(k));
                }
            };
            for (;;) {
                int item = atomicAdd(p.sched, 1);
                if (item >= total_items) item = -1;
                mbar_wait(sempty_bar(rs), rphase ^ 1u);
                ring[rs] = item;
                mbar_arrive(sfull_bar(rs));
                if (++rs == RING) { rs = 0; rphase ^= 1u; }
                if (item < 0) break;
                const int rt = item / M, e = item - rt * M;
                const int s = max(p.row_species[rt * BM], 0);
                const int se = s * M + e;
                const __half* w = p.wimg + (size_t)se * MID_W_TOTAL;
                {   // b2 | b3 | w4 of this network
                    mbar_wait(cempty_bar(cb), cphase ^ 1u);
                    const uint32_t dst = cst_s + (uint32_t)(cb * MID_CONST_BYTES);
                    mbar_expect_tx(cfull_bar(cb), (uint32_t)MID_CONST_BYTES);
                    bulk_load(dst, p.b2 + (size_t)se * H2, H2 * 4u, cfull_bar(cb));
                    bulk_load(dst + H2 * 4u, p.b3 + (size_t)se * H3, H3 * 4u, cfull_bar(cb));
                    bulk_load(dst + (H2 + H3) * 4u, p.w4 + (size_t)se * H3, H3 * 4u, cfull_bar(cb));
                    if (++cb == 2) { cb = 0; cphase ^= 1u; }
                }
                for (int j = 0; j < H1 / 32; ++j) {                       // G2: W2 K steps 2j, 2j+1 + the matching 32 columns of h1
                    // the ring's slots free up while the previous item's B2 runs; once they are refilled, wait for that B2
                    if (j == MID_SLOTS && prev_rt >= 0) load_h1_for_b2();
                    const uint32_t sa = next_slot();
                    mbar_expect_tx(full_bar(slot), MID_WB(64u * H2 * 2u) + 16384u);
                    bulk_load(sa, w + MID_W_G2 + (size_t)j * 64 * H2, MID_WB(64u * H2 * 2u), full_bar(slot));
                    const size_t goff = (size_t)((j & 1) * 4) * BM * 8;
                    bulk_load(sa + MID_A_OFF, p.h1 + tile_off(p.plane_tiles, M * 4, 0, rt, e * 4 + (j >> 1)) + goff, 8192u, full_bar(slot));
                    bulk_load(sa + MID_A_OFF + 8192, p.h1 + tile_off(p.plane_tiles, M * 4, 1, rt, e * 4 + (j >> 1)) + goff, 8192u,
                              full_bar(slot));
                    advance();
                }
                for (int j = 0; j < H2 / 32; ++j) {                       // G3
                    const uint32_t sa = next_slot();
                    mbar_expect_tx(full_bar(slot), MID_WB(64u * H3 * 2u));
                    bulk_load(sa, w + MID_W_G3 + (size_t)j * 64 * H3, MID_WB(64u * H3 * 2u), full_bar(slot));
                    advance();
                }
                if (p.forward_only) continue;
                for (int j = 0; j < H3 / 32; ++j) {                       // B3
                    const uint32_t sa = next_slot();
                    mbar_expect_tx(full_bar(slot), MID_WB(64u * H2 * 2u));
                    bulk_load(sa, w + MID_W_B3 + (size_t)j * 64 * H2, MID_WB(64u * H2 * 2u), full_bar(slot));
                    advance();
                }
                for (int j = 0; j < H2 / 32; ++j) {                       // B2
                    const uint32_t sa = next_slot();
                    mbar_expect_tx(full_bar(slot), MID_WB(64u * H1 * 2u));
                    bulk_load(sa, w + MID_W_B2 + (size_t)j * 64 * H1, MID_WB(64u * H1 * 2u), full_bar(slot));
                    advance();
                }
                prev_rt = rt; prev_e = e;
            }
            if (prev_rt >= 0) load_h1_for_b2();                          // the last item of this CTA
        }
    } else if (warp == MID_EPI_WARPS + 1) {
        // ===== MMA issuer =====
        // A source of a GEMM: the slot (G2: h1 streams in), X (G3: h2, B2: d2) or tensor memory (B3: d3).  A GEMM whose A is
        // produced by the previous epilogue waits for 64-column block kb of it (xr[kb]) before its K steps 4 kb .. 4 kb + 3.
        // Hazards, all covered by program order + these waits: a GEMM that overwrites an accumulator region is issued only
        // after every epilogue warp has signalled a block that it produces AFTER its last read of that region.
        if (elect_one()) {
            int slot = 0; uint32_t phase = 0;
            int rs = 0; uint32_t rphase = 0;
            uint32_t xphase = 0;                                   // bit k: parity of xr[k]
            int nit = 0; (void)nit;
            enum { A_SLOT = 0, A_X = 1, A_TMEM = 2 };
            auto run = [&](int n, int steps, int a_src, uint32_t d_tmem) {
                const uint32_t idesc = make_idesc(n);
                const uint32_t lbo_b = (uint32_t)n * 16u;
                uint32_t accumulate = 0u;
                for (int sl = 0; sl < steps / 2; ++sl) {                 // one ring slot = K steps 2 sl, 2 sl + 1
                    if (a_src != A_SLOT && (sl & 1) == 0) {
                        const int kb = sl >> 1;
                        mbar_wait(xr_bar(kb), (xphase >> kb) & 1u);
                        xphase ^= 1u << kb;
                        tc_fence_after();
                    }
                    mbar_wait(full_bar(slot), phase);
                    tc_fence_after();
                    const uint32_t sa = slots + (uint32_t)slot * MID_SLOT_BYTES;
#pragma unroll
                    for (int t = 0; t < 2; ++t) {
                        const int j = 2 * sl + t;
                        const uint32_t sb = sa + (uint32_t)t * 4u * lbo_b;
                        const uint64_t b_hi = make_desc_ns(sb, lbo_b), b_lo = make_desc_ns(sb + 2u * lbo_b, lbo_b);
                        if (!(MID_DBG & 2)) {
                            if (a_src == A_TMEM) {
                                const uint32_t a_hi = tmem_base + MID_D + (uint32_t)j * 8u, a_lo = tmem_base + MID_D_LO + (uint32_t)j * 8u;
                                umma_f16_ts(d_tmem, a_hi, b_hi, idesc, accumulate);
                                if (!p.single) {
                                    umma_f16_ts(d_tmem, a_hi, b_lo, idesc, 1u);
                                    umma_f16_ts(d_tmem, a_lo, b_hi, idesc, 1u);
                                }
                            } else {
                                const uint32_t a0 = a_src == A_SLOT ? sa + MID_A_OFF + (uint32_t)t * 4096u : xs + (uint32_t)j * 4096u;
                                const uint64_t a_hi = make_desc_ns(a0, 2048u);
                                const uint64_t a_lo = make_desc_ns(a0 + (a_src == A_SLOT ? 8192u : (uint32_t)MID_X_PLANE), 2048u);
                                umma_f16(d_tmem, a_hi, b_hi, idesc, accumulate);
                                if (!p.single) {
                                    umma_f16(d_tmem, a_hi, b_lo, idesc, 1u);
                                    umma_f16(d_tmem, a_lo, b_hi, idesc, 1u);
                                }
                            }
                        }
                        accumulate = 1u;
                    }
                    umma_commit(empty_bar(slot));
                    if (++slot == MID_SLOTS) { slot = 0; phase ^= 1u; }
                }
            };
            for (;;) {
                mbar_wait(sfull_bar(rs), rphase);
                const int item = ring[rs];
                mbar_arrive(sempty_bar(rs));
                if (++rs == RING) { rs = 0; rphase ^= 1u; }
                if (item < 0) break;
                TR(0, nit, 0);
                run(H2, H1 / 16, A_SLOT, tmem_base + MID_P); umma_commit(accp_bar);     // G2: h1 W2^T        -> P
                TR(0, nit, 1);
                run(H3, H2 / 16, A_X, tmem_base + MID_Q);    umma_commit(accq_bar);     // G3: h2 W3^T        -> Q
                TR(0, nit, 2);
                if (p.forward_only) continue;
                run(H2, H3 / 16, A_TMEM, tmem_base + MID_P); umma_commit(accp_bar);     // B3: d3 W3          -> P
                TR(0, nit, 3);
                run(H1, H2 / 16, A_X, tmem_base + MID_Q);    umma_commit(accq_bar);     // B2: d2 W2          -> Q u D
                umma_commit(xfree_bar);                                                  // ... and X is free for h1 (producer)
                TR(0, nit, 4);
                ++nit;
            }
        }
    } else {
        // ===== epilogue warps: a warp may touch only TMEM lanes 32 (warp % 4) .. + 31; the four warps of a lane
        //       quadrant take every fourth 16-column chunk, so round k of an epilogue covers columns 64 k .. 64 k + 63 =====
        const int q = warp & 3, cg = warp >> 2;
        const int r_in = q * 32 + lane;
        const uint32_t lane_base = tmem_base + ((uint32_t)(q * 32) << 16);
        int rs = 0; uint32_t rphase = 0;
        uint32_t pphase = 0, qphase = 0, hph = 0;
        int cb = 0; uint32_t cphase = 0;
        int nit = 0; (void)nit;
        const bool trw = warp == 0 && lane == 0; (void)trw;
        const float kexp = 1.4426950408889634f / p.alpha, inv_alpha = 1.0f / p.alpha;
        const float sc = 1.0f / W_SCALE;
        // this warp's part of 64-column block k is written (shared memory made visible to the tensor core's proxy, tensor
        // memory stores complete) and its accumulator reads of the round are done
        auto signal_x = [&](int k) {
            fence_proxy_async_smem();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(xr_bar(k));
        };
        auto signal_t = [&](int k) {                         // the same when the block went to tensor memory only
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(xr_bar(k));
        };
        auto lds16 = [&](const float* src, float (&x)[16]) {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const float4 t4 = *reinterpret_cast<const float4*>(src + 4 * i);
                x[4 * i] = t4.x; x[4 * i + 1] = t4.y; x[4 * i + 2] = t4.z; x[4 * i + 3] = t4.w;
            }
        };
        for (;;) {
            mbar_wait(sfull_bar(rs), rphase);
            const int item = ring[rs];
            __syncwarp();
            if (lane == 0) mbar_arrive(sempty_bar(rs));
            if (++rs == RING) { rs = 0; rphase ^= 1u; }
            if (item < 0) break;
            const int rt = item / M, e = item - rt * M;
            const int s = max(p.row_species[rt * BM], 0);
            const int row = rt * BM + r_in;
            const int se = s * M + e;
            uint32_t v[16];
            float x[16], aux[16];
            // the item's constants (b2 | b3 | w4) arrive in shared memory by bulk copy: no global load inside the rounds
            mbar_wait(cfull_bar(cb), cphase);
            const float* cst = cst_ptr + cb * MID_CONST_FLOATS;
            // ---- G2 (P): h2 = CELU(acc / 64 + b2) -> X, block by block
            if (trw) TR(1, nit, 0);
            mbar_wait(accp_bar, pphase); pphase ^= 1u;
            tc_fence_after();
            if (trw) TR(1, nit, 1);
#pragma unroll 1
            for (int k = 0; k < 3; ++k) {
                const int c0 = 64 * k + 16 * cg;
                if (!(MID_DBG & 1)) {
                    tmem_ld16_issue(lane_base + MID_P + (uint32_t)c0, v);
                    lds16(cst + c0, aux);
                    tmem_ld_wait();
#pragma unroll
                    for (int i = 0; i < 16; ++i) x[i] = celu_f(fmaf(__uint_as_float(v[i]), sc, aux[i]), p.alpha, kexp);
                    store_split16_x(x, x_ptr, c0, r_in);
                }
                signal_x(k);
                if (trw) TR(1, nit, 2 + k);
            }
            // ---- G3 (Q): h3 = CELU(acc / 64 + b3); E_i += (w4.h3 + b4)/M; d3 = w4 CELU'(z3) 2^10 / M -> tensor memory (A of B3)
            float w4v[16];
            mbar_wait(accq_bar, qphase); qphase ^= 1u;
            tc_fence_after();
            if (trw) TR(1, nit, 5);
            float e_acc = 0.f;
            const float dsc = p.inv_models * D_SCALE;
#pragma unroll 1
            for (int k = 0; k < 3; ++k) {
                const int c0 = 64 * k + 16 * cg;
                if (c0 < H3 && !(MID_DBG & 1)) {
                    tmem_ld16_issue(lane_base + MID_Q + (uint32_t)c0, v);
                    lds16(cst + H2 + c0, aux);
                    lds16(cst + H2 + H3 + c0, w4v);
                    tmem_ld_wait();
#pragma unroll
                    for (int i = 0; i < 16; ++i) {
                        const float h = celu_f(fmaf(__uint_as_float(v[i]), sc, aux[i]), p.alpha, kexp);
                        e_acc = fmaf(w4v[i], h, e_acc);
                        x[i] = w4v[i] * dsc * dcelu_from_h(h, inv_alpha);
                    }
                    if (!p.forward_only) {
                        uint32_t ph[8], pl[8];
#pragma unroll
                        for (int i = 0; i < 8; ++i) split_pair(x[2 * i], x[2 * i + 1], ph[i], pl[i]);   // K even -> low half
                        tmem_st8(lane_base + MID_D + (uint32_t)(c0 >> 1), ph);
                        tmem_st8(lane_base + MID_D_LO + (uint32_t)(c0 >> 1), pl);
                        tmem_st_wait();
                    }
                }
                if (!p.forward_only) signal_t(k);
                if (trw) TR(1, nit, 6 + k);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(cempty_bar(cb));                 // the constants buffer may be refilled
            if (++cb == 2) { cb = 0; cphase ^= 1u; }
            atomicAdd(&p.e_atom[row], (e_acc + (cg == 0 ? p.b4[se] : 0.f)) * p.inv_models);
            if (p.forward_only) { tc_fence_before(); continue; }
            // ---- B3 (P): d2 = (acc / 64) CELU'(z2), CELU' from this thread's own h2 in X, d2 written over it
            mbar_wait(accp_bar, pphase); pphase ^= 1u;
            tc_fence_after();
            if (trw) TR(1, nit, 9);
#pragma unroll 1
            for (int k = 0; k < 3; ++k) {
                const int c0 = 64 * k + 16 * cg;
                if (!(MID_DBG & 1)) {
                    tmem_ld16_issue(lane_base + MID_P + (uint32_t)c0, v);
                    uint4 hh[2], hl[2];
#pragma unroll
                    for (int i = 0; i < 2; ++i) {
                        const uint8_t* src = x_ptr + (size_t)(((c0 >> 3) + i) * BM + r_in) * 16;
                        hh[i] = *reinterpret_cast<const uint4*>(src);
                        hl[i] = *reinterpret_cast<const uint4*>(src + MID_X_PLANE);
                    }
                    join16(hh, hl, aux);
                    tmem_ld_wait();
#pragma unroll
                    for (int i = 0; i < 16; ++i) x[i] = __uint_as_float(v[i]) * sc * dcelu_from_h(aux[i], inv_alpha);
                    store_split16_x(x, x_ptr, c0, r_in);
                }
                signal_x(k);
                if (trw) TR(1, nit, 10 + k);
            }
            // ---- B2 (Q u D): d1 = (acc / 64) CELU'(z1) -> global (tiled planes).  CELU' needs the saved h1: its first three
            //      64-column blocks arrive in X by bulk copy once B2's MMAs are done with d2 (producer), the fourth by plain
            //      loads issued here, whose latency runs under the first three rounds
            uint4 gh[2], gl[2];
            auto h1_offsets = [&](int c0, size_t& o_hi, size_t& o_lo) {
                const size_t in_tile = (size_t)(((c0 & 63) >> 3) * BM + r_in) * 8;
                o_hi = tile_off(p.plane_tiles, M * 4, 0, rt, e * 4 + (c0 >> 6)) + in_tile;
                o_lo = tile_off(p.plane_tiles, M * 4, 1, rt, e * 4 + (c0 >> 6)) + in_tile;
            };
            uint4 lh[2], ll[2];
            if (!(MID_DBG & 1)) {
                size_t o_hi, o_lo;
                h1_offsets(192 + cg * 16, o_hi, o_lo);
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    lh[i] = *reinterpret_cast<const uint4*>(p.h1 + o_hi + i * (BM * 8));
                    ll[i] = *reinterpret_cast<const uint4*>(p.h1 + o_lo + i * (BM * 8));
                }
            }
            mbar_wait(accq_bar, qphase); qphase ^= 1u;
            tc_fence_after();
            if (trw) TR(1, nit, 13);
#pragma unroll 1
            for (int k = 0; k < 4 && !(MID_DBG & 1); ++k) {
                const int c0 = 64 * k + 16 * cg;
                tmem_ld16_issue(lane_base + MID_Q + (uint32_t)c0, v);
                if (k < 3) {
                    mbar_wait(hfull_bar(k), hph);
                    const uint8_t* src = x_ptr + (size_t)k * MID_H_ROUND + (size_t)((2 * cg) * BM + r_in) * 16;
#pragma unroll
                    for (int i = 0; i < 2; ++i) {
                        gh[i] = *reinterpret_cast<const uint4*>(src + i * (BM * 16));
                        gl[i] = *reinterpret_cast<const uint4*>(src + 16384 + i * (BM * 16));
                    }
                    join16(gh, gl, aux);
                } else {
                    join16(lh, ll, aux);
                }
                tmem_ld_wait();
#pragma unroll
                for (int i = 0; i < 16; ++i) x[i] = __uint_as_float(v[i]) * sc * dcelu_from_h(aux[i], inv_alpha);
                size_t o_hi, o_lo;
                h1_offsets(c0, o_hi, o_lo);
                if (!(MID_DBG & 4)) store_split16_tiled(x, p.d1 + o_hi, p.d1 + o_lo);
            }
            hph ^= 1u;
            tc_fence_before();
            // every epilogue warp has read its h1 out of X before any of them writes the next item's h2 into it
            asm volatile("bar.sync 1, %0;" ::"n"(32 * MID_EPI_WARPS) : "memory");
            if (trw) TR(1, nit, 14);
            ++nit;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == MID_EPI_WARPS + 1) tmem_dealloc(tmem_base, TMEM_COLS);
#if MID_TRACE
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        const long long t0 = g_tr[0][0][0];
        for (int it = 0; it < 8; ++it) {
            printf("MMA item %d:", it);
            for (int e = 0; e < 5; ++e) printf(" %lld", g_tr[0][it][e] - t0);
            printf("\nEPI item %d:", it);
            for (int e = 0; e < 15; ++e) printf(" %lld", g_tr[1][it][e] - t0);
            printf("\n");
        }
    }
#endif
}


// ======================================================================================================
// G1 fused into the front of the middle chain: one work item = (row tile, network) runs
//     AEV rows -> h1 -> h2 -> (E_i, d3) -> d2 -> d1
// inside one CTA, so h1 never goes to HBM as an operand (profiles/r2b: writing h1, 754 MB per step, is what G1 waited
// for, and reading it back was most of k_mlp_mid's first phase).  Differences from k_mlp_mid:
//   * G1 accumulates z1 (256 columns) in tensor memory; its epilogue writes h1 = CELU(z1 + b1) in 64-column blocks into X
//     as the A operand of G2 (the fourth block takes the place of the first once G2's first K block has been read), so G2
//     starts under G1's epilogue exactly as G3 starts under G2's.  The same thread also stores its h1 values to a per-CTA
//     scratch tile (128 KB, rewritten by every item: it stays in L2) from which B2's epilogue gets CELU'(z1) back.
//   * operands of G1 stream through the ring one 16-wide K step per slot: the W1 image of the step (16 KB, pre-tiled like
//     the other weights) and the AEV planes' 2 x 4 KB (tiled operand layout, aev_tiled_off()); only the feature blocks of the
//     row tile's mask are visited.
//   * tensor memory is used in a ping-pong map, offset O = 256 (item parity): z1 [O, O+256); G2 accumulator [O+256, O+448);
//     G3 accumulator [O, O+160); d3 [O+160, O+320) (hi 80 columns, lo 80 columns); B3 accumulator [O+320, O+512); B2
//     accumulator [O, O+256) - all modulo 512.  The next item's G1 (z1 at [O+256, ...)) therefore runs under this item's B2
//     epilogue, which is where the tensor pipe idled in k_mlp_mid while d1 was stored.
// ======================================================================================================
constexpr int FU_SLOTS = 5;
constexpr int FU_SLOT_BYTES = 24576;             // G1: W1 image of one K step (16 KB) + AEV hi (4 KB) + lo (4 KB); G2 / G3 / B3: two K steps; B2: one
constexpr int FU_A_OFF = 16384;
constexpr int FU_CONST_FLOATS = H1 + H2 + H3 + H3;   // b1 | b2 | b3 | w4
constexpr int FU_CONST_BYTES = FU_CONST_FLOATS * 4;
constexpr int FU_SMEM = MID_X_BYTES + FU_SLOTS * FU_SLOT_BYTES + 2 * FU_CONST_BYTES + 1024 /*align*/ + 512 /*barriers, TMEM word, ring*/;
static_assert(FU_SMEM <= 232448, "shared memory of k_mlp_fused");
constexpr int FU_W1_STEP = 32 * H1;              // halves of the W1 image of one K step: [plane][8-column group (2)][n][8]
constexpr int FU_SCRATCH = 2 * H1 * BM;          // halves of one CTA's h1 scratch tile: [plane][64-column block (4)][group][row][8]

struct FusedArgs {
    int single, forward_only, n_models, plane_tiles;
    const int* row_species;
    const int* sp_start;
    const unsigned* tile_mask;
    const __half* aev;        // AEV planes, tiled operand layout
    const __half* w1img;      // [species][network][64 K steps][FU_W1_STEP]
    const __half* wimg;       // [species][network][MID_W_TOTAL] (G2, G3, B3, B2)
    __half* scratch;          // [gridDim.x][FU_SCRATCH]
    __half* d1;
    const float *b1, *b2, *b3, *w4, *b4;
    float inv_models, alpha;
    float* e_atom;
    int* sched;
};

__device__ __forceinline__ void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }

__global__ void __launch_bounds__(MID_THREADS, 1)
k_mlp_fused(const FusedArgs p) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;
    uint8_t* x_ptr = smem_raw + (base - raw);
    const uint32_t xs = base;
    const uint32_t slots = base + MID_X_BYTES;
    const uint32_t cst_s = slots + FU_SLOTS * FU_SLOT_BYTES;
    const float* cst_ptr = reinterpret_cast<const float*>(x_ptr + MID_X_BYTES + FU_SLOTS * FU_SLOT_BYTES);
    const uint32_t bar0 = cst_s + 2 * FU_CONST_BYTES;
    uint64_t* bars = reinterpret_cast<uint64_t*>(x_ptr + MID_X_BYTES + FU_SLOTS * FU_SLOT_BYTES + 2 * FU_CONST_BYTES);
    // barriers: full[SLOTS], empty[SLOTS], then 17 single ones (below), sfull[RING], sempty[RING]; then the TMEM word and the item ring
    constexpr int NB1 = 18;   // acc1, accp, accq, xr[4], xfree[3], hfull[3], cfull[2], cempty[2], hsaved
    constexpr int NBARS = 2 * FU_SLOTS + NB1 + 2 * RING;
    auto full_bar = [&](int s) { return bar0 + 8u * s; };
    auto empty_bar = [&](int s) { return bar0 + 8u * (FU_SLOTS + s); };
    const uint32_t b1s = bar0 + 8u * (2 * FU_SLOTS);
    const uint32_t acc1_bar = b1s, accp_bar = b1s + 8u, accq_bar = b1s + 16u;
    auto xr_bar = [&](int k) { return b1s + 24u + 8u * k; };            // k = 0..3: 64-column block k of an epilogue's output is ready
    auto xfree_bar = [&](int k) { return b1s + 56u + 8u * k; };         // k = 0..2: B2 has read d2 block k: its place in X may take h1 block k back
    auto hfull_bar = [&](int k) { return b1s + 80u + 8u * k; };         // k = 0..2: h1 block k is back in X (for CELU'(z1))
    auto cfull_bar = [&](int b) { return b1s + 104u + 8u * b; };
    auto cempty_bar = [&](int b) { return b1s + 120u + 8u * b; };
    const uint32_t hsaved_bar = b1s + 136u;                             // plain-store variant: the item's h1 is in the scratch tile, visible to the async proxy
    auto sfull_bar = [&](int s) { return bar0 + 8u * (2 * FU_SLOTS + NB1 + s); };
    auto sempty_bar = [&](int s) { return bar0 + 8u * (2 * FU_SLOTS + NB1 + RING + s); };
    volatile uint32_t* tmem_word = reinterpret_cast<volatile uint32_t*>(bars + NBARS);
    volatile int* ring = reinterpret_cast<volatile int*>(bars + NBARS + 1);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int M = p.n_models;
    const int total_items = (p.sp_start[NSP] / BM) * M;
    __half* scratch = p.scratch + (size_t)blockIdx.x * FU_SCRATCH;

    if (warp == MID_EPI_WARPS && lane == 0) {
        for (int s = 0; s < FU_SLOTS; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
        mbar_init(acc1_bar, 1); mbar_init(accp_bar, 1); mbar_init(accq_bar, 1);
        for (int k = 0; k < 4; ++k) mbar_init(xr_bar(k), MID_EPI_WARPS);
        for (int k = 0; k < 3; ++k) { mbar_init(xfree_bar(k), 1); mbar_init(hfull_bar(k), 1); }
        mbar_init(hsaved_bar, MID_EPI_WARPS);
        for (int b = 0; b < 2; ++b) { mbar_init(cfull_bar(b), 1); mbar_init(cempty_bar(b), MID_EPI_WARPS); }
        for (int s = 0; s < RING; ++s) { mbar_init(sfull_bar(s), 1); mbar_init(sempty_bar(s), 1 + MID_EPI_WARPS); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == MID_EPI_WARPS + 1) tmem_alloc(smem_u32((const void*)tmem_word), TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_word;

    auto g1_mask = [&](int rt) -> unsigned { const unsigned m = p.tile_mask[rt]; return m ? m : (1u << 14); };   // an all-zero tile runs one block of zeros

    if (warp == MID_EPI_WARPS) {
        // ===== item scheduler + producer =====
        if (elect_one()) {
            int slot = 0; uint32_t phase = 0;
            int rs = 0; uint32_t rphase = 0;
            int cb = 0; uint32_t cphase = 0;
            uint32_t hphase = 0;
            bool have_prev = false;
            auto next_slot = [&]() -> uint32_t {
                mbar_wait(empty_bar(slot), phase ^ 1u);
                return slots + (uint32_t)slot * FU_SLOT_BYTES;
            };
            auto advance = [&]() { if (++slot == FU_SLOTS) { slot = 0; phase ^= 1u; } };
            // h1 of the PREVIOUS item: scratch -> X, block k as soon as that item's B2 has read d2 block k out of X (its K steps 4 k ..
            // 4 k + 3 have completed); three 64-column blocks (hi plane then lo plane) for CELU'(z1) in B2's epilogue, the fourth comes
            // by plain loads there.  The ring paces this thread by B2's progress (a G1 slot frees when a B2 step retires), so block 0
            // can go before the first G1 slot, block 1 after it and block 2 once the ring has been refilled: none of the waits blocks
            auto reload_h1 = [&](int k) {
                if (!FU_BULK_H1 && k == 0) mbar_wait(hsaved_bar, hphase);
                mbar_wait(xfree_bar(k), hphase);
                mbar_expect_tx(hfull_bar(k), (uint32_t)MID_H_ROUND);
                // (block k goes where d2's block k was: hi plane at 16 k KB, lo plane 48 KB further - nothing B2 still reads)
                bulk_load(xs + (uint32_t)k * 16384u, scratch + (size_t)k * (BM * BK), 16384u, hfull_bar(k));
                bulk_load(xs + (uint32_t)MID_X_PLANE + (uint32_t)k * 16384u, scratch + (size_t)(4 + k) * (BM * BK), 16384u, hfull_bar(k));
            };
            for (;;) {
                int item = atomicAdd(p.sched, 1);
                if (item >= total_items) item = -1;
                mbar_wait(sempty_bar(rs), rphase ^ 1u);
                ring[rs] = item;
                mbar_arrive(sfull_bar(rs));
                if (++rs == RING) { rs = 0; rphase ^= 1u; }
                if (item < 0) break;
                const int rt = item / M, e = item - rt * M;
                const int s = max(p.row_species[rt * BM], 0);
                const int se = s * M + e;
                const __half* w = p.wimg + (size_t)se * MID_W_TOTAL;
                const __half* w1 = p.w1img + (size_t)se * (AEV_LD / 16) * FU_W1_STEP;
                {   // b1 | b2 | b3 | w4 of this network
                    mbar_wait(cempty_bar(cb), cphase ^ 1u);
                    const uint32_t dst = cst_s + (uint32_t)(cb * FU_CONST_BYTES);
                    mbar_expect_tx(cfull_bar(cb), (uint32_t)FU_CONST_BYTES);
                    bulk_load(dst, p.b1 + (size_t)se * H1, H1 * 4u, cfull_bar(cb));
                    bulk_load(dst + H1 * 4u, p.b2 + (size_t)se * H2, H2 * 4u, cfull_bar(cb));
                    bulk_load(dst + (H1 + H2) * 4u, p.b3 + (size_t)se * H3, H3 * 4u, cfull_bar(cb));
                    bulk_load(dst + (H1 + H2 + H3) * 4u, p.w4 + (size_t)se * H3, H3 * 4u, cfull_bar(cb));
                    if (++cb == 2) { cb = 0; cphase ^= 1u; }
                }
                // G1: the K steps of the active feature blocks.  The ring refills while the previous item's B2 runs; once it is
                // full, wait for that B2 and bring the previous item's h1 back for its epilogue
                int next_reload = (!have_prev || p.forward_only) ? 3 : 0;
                int issued = 0;
                for (unsigned km = g1_mask(rt); km; km &= km - 1u) {
                    const int kb = __ffs(km) - 1;
                    const __half* a_hi = p.aev + tile_off(p.plane_tiles, N_KBLK, 0, rt, kb);
                    const __half* a_lo = p.aev + tile_off(p.plane_tiles, N_KBLK, 1, rt, kb);
                    for (int ks = 0; ks < 4; ++ks) {
                        if (next_reload < 3 && (issued == 0 || issued == 1 || issued == FU_SLOTS)) reload_h1(next_reload++);
                        const uint32_t sa = next_slot();
                        mbar_expect_tx(full_bar(slot), (uint32_t)FU_SLOT_BYTES);
                        bulk_load(sa, w1 + (size_t)(kb * 4 + ks) * FU_W1_STEP, 16384u, full_bar(slot));
                        bulk_load(sa + FU_A_OFF, a_hi + ks * (2 * BM * 8), 4096u, full_bar(slot));
                        bulk_load(sa + FU_A_OFF + 4096u, a_lo + ks * (2 * BM * 8), 4096u, full_bar(slot));
                        advance();
                        ++issued;
                    }
                }
                while (next_reload < 3) reload_h1(next_reload++);
                if (have_prev && !p.forward_only) hphase ^= 1u;
                for (int j = 0; j < H1 / 32; ++j) {                       // G2: W2 K steps 2j, 2j+1 (A = h1 in X)
                    const uint32_t sa = next_slot();
                    mbar_expect_tx(full_bar(slot), 64u * H2 * 2u);
                    bulk_load(sa, w + MID_W_G2 + (size_t)j * 64 * H2, 64u * H2 * 2u, full_bar(slot));
                    advance();
                }
                for (int j = 0; j < H2 / 32; ++j) {                       // G3
                    const uint32_t sa = next_slot();
                    mbar_expect_tx(full_bar(slot), 64u * H3 * 2u);
                    bulk_load(sa, w + MID_W_G3 + (size_t)j * 64 * H3, 64u * H3 * 2u, full_bar(slot));
                    advance();
                }
                have_prev = true;
                if (p.forward_only) continue;
                for (int j = 0; j < H3 / 32; ++j) {                       // B3
                    const uint32_t sa = next_slot();
                    mbar_expect_tx(full_bar(slot), 64u * H2 * 2u);
                    bulk_load(sa, w + MID_W_B3 + (size_t)j * 64 * H2, 64u * H2 * 2u, full_bar(slot));
                    advance();
                }
                for (int j = 0; j < H2 / 16; ++j) {                       // B2: one K step per slot (16 KB)
                    const uint32_t sa = next_slot();
                    mbar_expect_tx(full_bar(slot), 32u * H1 * 2u);
                    bulk_load(sa, w + MID_W_B2 + (size_t)j * 32 * H1, 32u * H1 * 2u, full_bar(slot));
                    advance();
                }
            }
            if (have_prev && !p.forward_only) for (int k = 0; k < 3; ++k) reload_h1(k);   // the last item of this CTA
        }
    } else if (warp == MID_EPI_WARPS + 1) {
        // ===== MMA issuer =====
        if (elect_one()) {
            int slot = 0; uint32_t phase = 0;
            int rs = 0; uint32_t rphase = 0;
            uint32_t xphase = 0;                                   // bit k: parity of xr[k]
            int nit = 0;
            auto wait_xr = [&](int kb) {
                mbar_wait(xr_bar(kb), (xphase >> kb) & 1u);
                xphase ^= 1u << kb;
                tc_fence_after();
            };
            auto wait_slot = [&]() -> uint32_t {
                mbar_wait(full_bar(slot), phase);
                tc_fence_after();
                return slots + (uint32_t)slot * FU_SLOT_BYTES;
            };
            auto release_slot = [&]() {
                umma_commit(empty_bar(slot));
                if (++slot == FU_SLOTS) { slot = 0; phase ^= 1u; }
            };
            auto mma3 = [&](uint32_t d, uint64_t a_hi, uint64_t a_lo, uint64_t b_hi, uint64_t b_lo, uint32_t idesc, uint32_t acc) {
                umma_f16(d, a_hi, b_hi, idesc, acc);
                if (!p.single) { umma_f16(d, a_hi, b_lo, idesc, 1u); umma_f16(d, a_lo, b_hi, idesc, 1u); }
            };
            auto mma3_ts = [&](uint32_t d, uint32_t a_hi, uint32_t a_lo, uint64_t b_hi, uint64_t b_lo, uint32_t idesc, uint32_t acc) {
                umma_f16_ts(d, a_hi, b_hi, idesc, acc);
                if (!p.single) { umma_f16_ts(d, a_hi, b_lo, idesc, 1u); umma_f16_ts(d, a_lo, b_hi, idesc, 1u); }
            };
            for (;;) {
                mbar_wait(sfull_bar(rs), rphase);
                const int item = ring[rs];
                mbar_arrive(sempty_bar(rs));
                if (++rs == RING) { rs = 0; rphase ^= 1u; }
                if (item < 0) break;
                const int rt = item / M;
                const uint32_t O = (nit & 1) ? 256u : 0u;
                TR(0, nit, 0);
                {   // G1: AEV W1^T -> z1 at [O, O + 256)
                    const uint32_t idesc = make_idesc(H1);
                    const int nsteps = 4 * __popc(g1_mask(rt));
#if MID_TRACE
                    if (blockIdx.x == 0 && nit >= 8 && nit < 16) g_tr[2][nit - 8][0] = nsteps;
#endif
                    uint32_t accumulate = 0u;
                    for (int j = 0; j < nsteps; ++j) {
                        const uint32_t sa = wait_slot();
                        mma3(tmem_base + O, make_desc_ns(sa + FU_A_OFF, 2048u), make_desc_ns(sa + FU_A_OFF + 4096u, 2048u),
                             make_desc_ns(sa, H1 * 16u), make_desc_ns(sa + 2u * H1 * 16u, H1 * 16u), idesc, accumulate);
                        accumulate = 1u;
                        release_slot();
                    }
                    umma_commit(acc1_bar);
                }
                TR(0, nit, 1);
                {   // G2: h1 W2^T -> [O + 256, O + 448); h1 block kb is K steps 4 kb .. 4 kb + 3: blocks 0..2 in X, block 3 in tensor memory
                    const uint32_t idesc = make_idesc(H2), lbo = H2 * 16u, d = tmem_base + (O ^ 256u);
                    uint32_t accumulate = 0u;
                    for (int sl = 0; sl < H1 / 32; ++sl) {
                        if ((sl & 1) == 0) {
                            const int kb = sl >> 1;
                            wait_xr(kb);
                            if (FU_BULK_H1 && kb < 3 && !p.forward_only) {      // h1 block kb (every epilogue warp has fenced its part) -> scratch tile
                                bulk_store(scratch + (size_t)kb * (BM * BK), xs + (uint32_t)kb * 16384u, 16384u);
                                bulk_store(scratch + (size_t)(4 + kb) * (BM * BK), xs + (uint32_t)MID_X_PLANE + (uint32_t)kb * 16384u, 16384u);
                                bulk_commit();
                            }
                        }
                        const uint32_t sa = wait_slot();
#pragma unroll
                        for (int t = 0; t < 2; ++t) {
                            const int j = 2 * sl + t;
                            const uint32_t sb = sa + (uint32_t)t * 4u * lbo;
                            if (j < 12) {
                                const uint32_t a0 = xs + (uint32_t)j * 4096u;
                                mma3(d, make_desc_ns(a0, 2048u), make_desc_ns(a0 + (uint32_t)MID_X_PLANE, 2048u), make_desc_ns(sb, lbo),
                                     make_desc_ns(sb + 2u * lbo, lbo), idesc, accumulate);
                            } else {                                      // block 3 of h1 is in tensor memory: hi [O + 448, + 32), lo [O + 480, + 32)
                                const uint32_t a_hi = tmem_base + ((O + 448u + 8u * (uint32_t)(j - 12)) & 511u);
                                mma3_ts(d, a_hi, a_hi + 32u, make_desc_ns(sb, lbo), make_desc_ns(sb + 2u * lbo, lbo), idesc, accumulate);
                            }
                            accumulate = 1u;
                        }
                        release_slot();
                    }
                    if (FU_BULK_H1) bulk_wait_all();                      // blocks 0..2 have left X (G2's epilogue overwrites them) and are in the scratch tile
                    umma_commit(accp_bar);
                }
                TR(0, nit, 2);
                {   // G3: h2 W3^T -> [O, O + 160)
                    const uint32_t idesc = make_idesc(H3), lbo = H3 * 16u, d = tmem_base + O;
                    uint32_t accumulate = 0u;
                    for (int sl = 0; sl < H2 / 32; ++sl) {
                        if ((sl & 1) == 0) wait_xr(sl >> 1);
                        const uint32_t sa = wait_slot();
#pragma unroll
                        for (int t = 0; t < 2; ++t) {
                            const int j = 2 * sl + t;
                            const uint32_t sb = sa + (uint32_t)t * 4u * lbo;
                            const uint32_t a0 = xs + (uint32_t)j * 4096u;
                            mma3(d, make_desc_ns(a0, 2048u), make_desc_ns(a0 + (uint32_t)MID_X_PLANE, 2048u), make_desc_ns(sb, lbo),
                                 make_desc_ns(sb + 2u * lbo, lbo), idesc, accumulate);
                            accumulate = 1u;
                        }
                        release_slot();
                    }
                    umma_commit(accq_bar);
                }
                TR(0, nit, 3);
                if (p.forward_only) { ++nit; continue; }
                {   // B3: d3 W3 -> [O + 320, O + 512); A = d3 in tensor memory, K step j at hi (O + 160 + 8 j), lo (O + 240 + 8 j) mod 512
                    const uint32_t idesc = make_idesc(H2), lbo = H2 * 16u, d = tmem_base + ((O + 320u) & 511u);
                    uint32_t accumulate = 0u;
                    for (int sl = 0; sl < H3 / 32; ++sl) {
                        if ((sl & 1) == 0) wait_xr(sl >> 1);
                        const uint32_t sa = wait_slot();
#pragma unroll
                        for (int t = 0; t < 2; ++t) {
                            const uint32_t j = (uint32_t)(2 * sl + t);
                            const uint32_t sb = sa + (uint32_t)t * 4u * lbo;
                            mma3_ts(d, tmem_base + ((O + 160u + 8u * j) & 511u), tmem_base + ((O + 240u + 8u * j) & 511u), make_desc_ns(sb, lbo),
                                    make_desc_ns(sb + 2u * lbo, lbo), idesc, accumulate);
                            accumulate = 1u;
                        }
                        release_slot();
                    }
                    umma_commit(accp_bar);
                }
                TR(0, nit, 4);
                {   // B2: d2 W2 -> [O, O + 256); one K step per slot
                    const uint32_t idesc = make_idesc(H1), lbo = H1 * 16u, d = tmem_base + O;
                    uint32_t accumulate = 0u;
                    for (int j = 0; j < H2 / 16; ++j) {
                        if ((j & 3) == 0) wait_xr(j >> 2);
                        const uint32_t sa = wait_slot();
                        const uint32_t a0 = xs + (uint32_t)j * 4096u;
                        mma3(d, make_desc_ns(a0, 2048u), make_desc_ns(a0 + (uint32_t)MID_X_PLANE, 2048u), make_desc_ns(sa, lbo),
                             make_desc_ns(sa + 2u * lbo, lbo), idesc, accumulate);
                        accumulate = 1u;
                        release_slot();
                        if ((j & 3) == 3) umma_commit(xfree_bar(j >> 2)); // d2 block j / 4 has been read: its place is free for the h1 reload (producer)
                    }
                    umma_commit(accq_bar);
                }
                TR(0, nit, 5);
                ++nit;
            }
        }
    } else {
        // ===== epilogue warps: a warp may touch only TMEM lanes 32 (warp % 4) .. + 31; the four warps of a lane
        //       quadrant take every fourth 16-column chunk, so round k of an epilogue covers columns 64 k .. 64 k + 63 =====
        const int q = warp & 3, cg = warp >> 2;
        const int r_in = q * 32 + lane;
        const uint32_t lane_base = tmem_base + ((uint32_t)(q * 32) << 16);
        int rs = 0; uint32_t rphase = 0;
        uint32_t a1phase = 0, pphase = 0, qphase = 0, hph = 0;
        int cb = 0; uint32_t cphase = 0;
        int nit = 0;
        const float kexp = 1.4426950408889634f / p.alpha, inv_alpha = 1.0f / p.alpha;
        const float sc = 1.0f / W_SCALE;
        auto signal_x = [&](int k) {
            fence_proxy_async_smem();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(xr_bar(k));
        };
        auto signal_t = [&](int k) {
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(xr_bar(k));
        };
        auto lds16 = [&](const float* src, float (&x)[16]) {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const float4 t4 = *reinterpret_cast<const float4*>(src + 4 * i);
                x[4 * i] = t4.x; x[4 * i + 1] = t4.y; x[4 * i + 2] = t4.z; x[4 * i + 3] = t4.w;
            }
        };
        // this thread's 16 columns c0.. of the scratch tile / of d1's item: offsets inside one plane of 4 blocks
        auto tile_in = [&](int c0) -> size_t { return (size_t)(c0 >> 6) * (BM * BK) + (size_t)(((c0 & 63) >> 3) * BM + r_in) * 8; };
        for (;;) {
            mbar_wait(sfull_bar(rs), rphase);
            const int item = ring[rs];
            __syncwarp();
            if (lane == 0) mbar_arrive(sempty_bar(rs));
            if (++rs == RING) { rs = 0; rphase ^= 1u; }
            if (item < 0) break;
            const int rt = item / M, e = item - rt * M;
            const int s = max(p.row_species[rt * BM], 0);
            const int row = rt * BM + r_in;
            const int se = s * M + e;
            const uint32_t O = (nit & 1) ? 256u : 0u;
            const bool trw = warp == 0 && lane == 0; (void)trw;
            uint32_t v[16];
            float x[16], aux[16];
            mbar_wait(cfull_bar(cb), cphase);
            const float* cst = cst_ptr + cb * FU_CONST_FLOATS;
            // ---- G1 (z1): h1 = CELU(acc / 64 + b1) -> X (A of G2) and, for CELU'(z1) later, the scratch tile
            if (trw) TR(1, nit, 0);
            mbar_wait(acc1_bar, a1phase); a1phase ^= 1u;
            tc_fence_after();
            if (trw) TR(1, nit, 1);
#pragma unroll 1
            for (int k = 0; k < 4; ++k) {
                const int c0 = 64 * k + 16 * cg;
                tmem_ld16_issue(lane_base + O + (uint32_t)c0, v);
                lds16(cst + c0, aux);
                tmem_ld_wait();
                celu16(v, aux, sc, p.alpha, kexp, x);
                if (k < 3) {
                    store_split16_x(x, x_ptr, c0, r_in);
                    signal_x(k);
                    if (!FU_BULK_H1 && !p.forward_only) {      // ... and to the scratch tile, after the signal: G2 does not wait for these stores
                        store_split16_tiled(x, scratch + tile_in(c0), scratch + (size_t)4 * (BM * BK) + tile_in(c0));
                    }
                } else {                     // X holds three blocks: the fourth is G2's A operand from tensor memory (the 64 columns no accumulator uses)
                    uint32_t ph[8], pl[8];
#pragma unroll
                    for (int i = 0; i < 8; ++i) split_pair(x[2 * i], x[2 * i + 1], ph[i], pl[i]);   // K even -> low half
                    tmem_st8(lane_base + ((O + 448u + 8u * (uint32_t)cg) & 511u), ph);
                    tmem_st8(lane_base + ((O + 480u + 8u * (uint32_t)cg) & 511u), pl);
                    tmem_st_wait();
                    signal_t(k);
                }
                // blocks 0..2 go to the scratch tile as bulk copies out of X (MMA issuer); block 3, which B2's epilogue reads back with
                // plain loads, is stored by the thread that will read it
                if (k == 3 && !p.forward_only) store_split16_tiled(x, scratch + tile_in(c0), scratch + (size_t)4 * (BM * BK) + tile_in(c0));
                if (trw) TR(1, nit, 2 + k);
            }
            if (!FU_BULK_H1 && !p.forward_only) {       // this warp's scratch stores are ordered before the producer's bulk reads
                fence_proxy_async_all();
                __syncwarp();
                if (lane == 0) mbar_arrive(hsaved_bar);
            }
            // ---- G2: h2 = CELU(acc / 64 + b2) -> X, block by block
            mbar_wait(accp_bar, pphase); pphase ^= 1u;
            tc_fence_after();
            if (trw) TR(1, nit, 6);
#pragma unroll 1
            for (int k = 0; k < 3; ++k) {
                const int c0 = 64 * k + 16 * cg;
                tmem_ld16_issue(lane_base + (O ^ 256u) + (uint32_t)c0, v);
                lds16(cst + H1 + c0, aux);
                tmem_ld_wait();
                celu16(v, aux, sc, p.alpha, kexp, x);
                store_split16_x(x, x_ptr, c0, r_in);
                signal_x(k);
                if (trw) TR(1, nit, 7 + k);
            }
            // ---- G3: h3 = CELU(acc / 64 + b3); E_i += (w4.h3 + b4)/M; d3 = w4 CELU'(z3) 2^10 / M -> tensor memory (A of B3)
            float w4v[16];
            mbar_wait(accq_bar, qphase); qphase ^= 1u;
            tc_fence_after();
            if (trw) TR(1, nit, 10);
            float e_acc = 0.f;
            const float dsc = p.inv_models * D_SCALE;
#pragma unroll 1
            for (int k = 0; k < 3; ++k) {
                const int c0 = 64 * k + 16 * cg;
                if (c0 < H3) {
                    tmem_ld16_issue(lane_base + O + (uint32_t)c0, v);
                    lds16(cst + H1 + H2 + c0, aux);
                    lds16(cst + H1 + H2 + H3 + c0, w4v);
                    tmem_ld_wait();
                    float h3[16];
                    celu16(v, aux, sc, p.alpha, kexp, h3);
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        float g0, g1;
                        e_acc = fmaf(w4v[2 * i], h3[2 * i], e_acc);
                        e_acc = fmaf(w4v[2 * i + 1], h3[2 * i + 1], e_acc);
                        unpack2(fma2(pack2(h3[2 * i], h3[2 * i + 1]), pack2(inv_alpha, inv_alpha), pack2(1.0f, 1.0f)), g0, g1);
                        unpack2(mul2(mul2(pack2(w4v[2 * i], w4v[2 * i + 1]), pack2(dsc, dsc)), pack2(fminf(g0, 1.0f), fminf(g1, 1.0f))), x[2 * i], x[2 * i + 1]);
                    }
                    if (!p.forward_only) {
                        uint32_t ph[8], pl[8];
#pragma unroll
                        for (int i = 0; i < 8; ++i) split_pair(x[2 * i], x[2 * i + 1], ph[i], pl[i]);   // K even -> low half
                        tmem_st8(lane_base + ((O + 160u + (uint32_t)(c0 >> 1)) & 511u), ph);
                        tmem_st8(lane_base + ((O + 240u + (uint32_t)(c0 >> 1)) & 511u), pl);
                        tmem_st_wait();
                    }
                }
                if (!p.forward_only) signal_t(k);
                if (trw) TR(1, nit, 11 + k);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(cempty_bar(cb));
            if (++cb == 2) { cb = 0; cphase ^= 1u; }
            atomicAdd(&p.e_atom[row], (e_acc + (cg == 0 ? p.b4[se] : 0.f)) * p.inv_models);
            if (p.forward_only) { tc_fence_before(); ++nit; continue; }
            // ---- B3: d2 = (acc / 64) CELU'(z2), CELU' from this thread's own h2 in X, d2 written over it
            mbar_wait(accp_bar, pphase); pphase ^= 1u;
            tc_fence_after();
            if (trw) TR(1, nit, 14);
#pragma unroll 1
            for (int k = 0; k < 3; ++k) {
                const int c0 = 64 * k + 16 * cg;
                tmem_ld16_issue(lane_base + ((O + 320u) & 511u) + (uint32_t)c0, v);
                uint4 hh[2], hl[2];
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    const uint8_t* src = x_ptr + (size_t)(((c0 >> 3) + i) * BM + r_in) * 16;
                    hh[i] = *reinterpret_cast<const uint4*>(src);
                    hl[i] = *reinterpret_cast<const uint4*>(src + MID_X_PLANE);
                }
                join16(hh, hl, aux);
                tmem_ld_wait();
                dcelu16(v, aux, sc, inv_alpha, x);
                store_split16_x(x, x_ptr, c0, r_in);
                signal_x(k);
                if (trw) TR(1, nit, 15 + k);
            }
            // ---- B2: d1 = (acc / 64) CELU'(z1) -> global (tiled planes).  h1 blocks 0..2 come back into X by bulk copy (producer),
            //      block 3 by plain loads of what this very thread stored (issued here, their latency runs under the first rounds)
            uint4 gh[2], gl[2], lh[2], ll[2];
            {
                const __half* s_hi = scratch + tile_in(192 + cg * 16);
                const __half* s_lo = s_hi + (size_t)4 * (BM * BK);
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    lh[i] = *reinterpret_cast<const uint4*>(s_hi + i * (BM * 8));
                    ll[i] = *reinterpret_cast<const uint4*>(s_lo + i * (BM * 8));
                }
            }
            mbar_wait(accq_bar, qphase); qphase ^= 1u;
            tc_fence_after();
            if (trw) TR(1, nit, 18);
            __half* d_hi = p.d1 + tile_off(p.plane_tiles, M * 4, 0, rt, e * 4);
            __half* d_lo = p.d1 + tile_off(p.plane_tiles, M * 4, 1, rt, e * 4);
#pragma unroll 1
            for (int k = 0; k < 4; ++k) {
                const int c0 = 64 * k + 16 * cg;
                tmem_ld16_issue(lane_base + O + (uint32_t)c0, v);
                if (k < 3) {
                    mbar_wait(hfull_bar(k), hph);
                    const uint8_t* src = x_ptr + (size_t)k * 16384 + (size_t)((2 * cg) * BM + r_in) * 16;
#pragma unroll
                    for (int i = 0; i < 2; ++i) {
                        gh[i] = *reinterpret_cast<const uint4*>(src + i * (BM * 16));
                        gl[i] = *reinterpret_cast<const uint4*>(src + MID_X_PLANE + i * (BM * 16));
                    }
                    join16(gh, gl, aux);
                } else {
                    join16(lh, ll, aux);
                }
                tmem_ld_wait();
                dcelu16(v, aux, sc, inv_alpha, x);
                if (FU_BULK_D1 && k < 3) {
                    // d1 over this thread's own h1 in X (already the global tiled layout of the block), then the block leaves as two
                    // bulk copies: 3/4 of d1 never passes through the LSU store path
                    uint8_t* dst = x_ptr + (size_t)k * 16384 + (size_t)((2 * cg) * BM + r_in) * 16;
                    uint32_t ph[8], pl[8];
#pragma unroll
                    for (int i = 0; i < 8; ++i) split_pair(x[2 * i], x[2 * i + 1], ph[i], pl[i]);
#pragma unroll
                    for (int i = 0; i < 2; ++i) {
                        *reinterpret_cast<uint4*>(dst + i * (BM * 16)) = make_uint4(ph[4 * i], ph[4 * i + 1], ph[4 * i + 2], ph[4 * i + 3]);
                        *reinterpret_cast<uint4*>(dst + MID_X_PLANE + i * (BM * 16)) = make_uint4(pl[4 * i], pl[4 * i + 1], pl[4 * i + 2], pl[4 * i + 3]);
                    }
                    fence_proxy_async_smem();
                    asm volatile("bar.sync 2, %0;" ::"n"(32 * MID_EPI_WARPS) : "memory");
                    if (warp == 0 && lane == 0) {
                        bulk_store(d_hi + (size_t)k * (BM * BK), xs + (uint32_t)k * 16384u, 16384u);
                        bulk_store(d_lo + (size_t)k * (BM * BK), xs + (uint32_t)MID_X_PLANE + (uint32_t)k * 16384u, 16384u);
                        bulk_commit();
                    }
                } else {
                    store_split16_tiled(x, d_hi + tile_in(c0), d_lo + tile_in(c0));
                }
                if (trw) TR(1, nit, 19 + k);
            }
            hph ^= 1u;
            if (FU_BULK_D1 && warp == 0 && lane == 0) bulk_wait_read<0>();       // d1's blocks have left X
            tc_fence_before();
            // every epilogue warp has read its h1 out of X before any of them writes the next item's h1 into it
            asm volatile("bar.sync 1, %0;" ::"n"(32 * MID_EPI_WARPS) : "memory");
            if (trw) TR(1, nit, 23);
            ++nit;
        }
    }
    if (threadIdx.x == 0) bulk_wait_all();
    tc_fence_before();
    __syncthreads();
    if (warp == MID_EPI_WARPS + 1) tmem_dealloc(tmem_base, TMEM_COLS);
#if MID_TRACE
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        const long long t0 = g_tr[0][0][0];
        for (int it = 0; it < 8; ++it) {
            printf("FMMA item %d (%lld G1 steps):", it, g_tr[2][it][0]);
            for (int e = 0; e < 6; ++e) printf(" %lld", g_tr[0][it][e] - t0);
            printf("\nFEPI item %d:", it);
            for (int e = 0; e < 24; ++e) printf(" %lld", g_tr[1][it][e] - t0);
            printf("\n");
        }
    }
#endif
}

// W1 images for k_mlp_fused: img[(s*M + e)][K step (64)][plane][8-column group (2)][n (256)][8], columns in the internal AEV order
__global__ void k_prep_w1img(const float* __restrict__ blob, int n_models, __half* __restrict__ img) {
    const int se = blockIdx.y;
    const int s = se / n_models, e = se - s * n_models;
    const float* net = blob + (size_t)(e * NSP + s) * NET_PARAMS;
    const int total = (AEV_LD / 16) * FU_W1_STEP;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        const int step = idx / FU_W1_STEP;
        int rem = idx - step * FU_W1_STEP;
        const int plane = rem / (16 * H1);
        rem -= plane * 16 * H1;
        const int g = rem / (8 * H1);
        rem -= g * 8 * H1;
        const int n = rem >> 3, c = 16 * step + 8 * g + (rem & 7);
        const int k = col2feat(c);
        const float v = k >= 0 ? net[OFF_W1 + (size_t)n * AEV_DIM + k] : 0.f;
        __half hi, lo;
        split_half(v * W_SCALE, hi, lo);
        img[(size_t)se * total + idx] = plane ? lo : hi;
    }
}

// weight images for k_mlp_mid: img[(s*M + e)][MID_W_TOTAL], see the layout above
__global__ void k_prep_mid(const float* __restrict__ blob, int n_models, __half* __restrict__ img) {
    const int se = blockIdx.y;                      // s * n_models + e
    const int s = se / n_models, e = se - s * n_models;
    const float* net = blob + (size_t)(e * NSP + s) * NET_PARAMS;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < MID_W_TOTAL; idx += gridDim.x * blockDim.x) {
        int n_rows, rem, mode;
        if (idx < MID_W_G3) { mode = 0; n_rows = H2; rem = idx - MID_W_G2; }
        else if (idx < MID_W_B3) { mode = 1; n_rows = H3; rem = idx - MID_W_G3; }
        else if (idx < MID_W_B2) { mode = 2; n_rows = H2; rem = idx - MID_W_B3; }
        else { mode = 3; n_rows = H1; rem = idx - MID_W_B2; }
        const int step = rem / (32 * n_rows);
        rem -= step * 32 * n_rows;
        const int plane = rem / (16 * n_rows);
        rem -= plane * 16 * n_rows;
        const int g = rem / (8 * n_rows);
        rem -= g * 8 * n_rows;
        const int n = rem >> 3, k = 16 * step + 8 * g + (rem & 7);
        float v;
        switch (mode) {
            case 0: v = net[OFF_W2 + n * H1 + k]; break;       // B(n,k) = W2[n][k]
            case 1: v = net[OFF_W3 + n * H2 + k]; break;       // W3[n][k]
            case 2: v = net[OFF_W3 + k * H2 + n]; break;       // W3[k][n]
            default: v = net[OFF_W2 + k * H1 + n]; break;      // W2[k][n]
        }
        __half hi, lo;
        split_half(v * W_SCALE, hi, lo);
        img[(size_t)se * MID_W_TOTAL + idx] = plane ? lo : hi;
    }
}

// ---- operand preparation -------------------------------------------------------------------------------
// fp32 rows -> hi / lo fp16 planes (AEV rows for G1)
__global__ void k_split_rows(const float* __restrict__ src, int ld_src, const int* __restrict__ sp_start, int ncol,
                             __half* __restrict__ dst, int plane_rows) {
    const int rows = sp_start[NSP];
    const size_t total = (size_t)rows * (ncol / 4);
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        const int r = (int)(idx / (ncol / 4)), c = (int)(idx % (ncol / 4)) * 4;
        const float4 v = *reinterpret_cast<const float4*>(src + (size_t)r * ld_src + c);
        __half h[4], l[4];
        split_half(v.x, h[0], l[0]); split_half(v.y, h[1], l[1]); split_half(v.z, h[2], l[2]); split_half(v.w, h[3], l[3]);
        // the tiled operand layout of the AEV planes (ncol = AEV_LD): 4 consecutive columns stay inside one 8-column group
        *reinterpret_cast<uint2*>(dst + aev_tiled_off(r, c)) = *reinterpret_cast<uint2*>(h);
        *reinterpret_cast<uint2*>(dst + (size_t)plane_rows * ncol + aev_tiled_off(r, c)) = *reinterpret_cast<uint2*>(l);
    }
}

// weight tiles: dst[(2*s + plane)*rows + r][c] = split(W_SCALE * src(r, c)); see the modes below
enum { WP_W1F = 0, WP_W2F, WP_W3F, WP_W3B, WP_W2B, WP_W1B };
__global__ void k_prep_weights(const float* __restrict__ blob, int n_models, int mode, int rows, int cols, __half* __restrict__ dst) {
    const int s = blockIdx.y;
    const size_t total = (size_t)rows * cols;
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        const int r = (int)(idx / cols), c = (int)(idx % cols);
        float v = 0.f;
        int e, n, k;
        switch (mode) {
            case WP_W1F: e = r / H1; n = r % H1; k = col2feat(c);       // columns in the internal AEV order
                if (k >= 0) v = blob[(size_t)(e * NSP + s) * NET_PARAMS + OFF_W1 + (size_t)n * AEV_DIM + k]; break;
            case WP_W2F: e = r / H2; n = r % H2; k = c;
                v = blob[(size_t)(e * NSP + s) * NET_PARAMS + OFF_W2 + n * H1 + k]; break;
            case WP_W3F: e = r / H3; n = r % H3; k = c;
                v = blob[(size_t)(e * NSP + s) * NET_PARAMS + OFF_W3 + n * H2 + k]; break;
            case WP_W3B: e = r / H2; n = r % H2; k = c;          // B(n,k) = W3[k][n]
                v = blob[(size_t)(e * NSP + s) * NET_PARAMS + OFF_W3 + k * H2 + n]; break;
            case WP_W2B: e = r / H1; n = r % H1; k = c;          // B(n,k) = W2[k][n]
                v = blob[(size_t)(e * NSP + s) * NET_PARAMS + OFF_W2 + k * H1 + n]; break;
            default: n = col2feat(r); e = c / H1; k = c % H1;    // WP_W1B: B(n, e*256+j) = W1_e[j][feature of column n]
                if (n >= 0) v = blob[(size_t)(e * NSP + s) * NET_PARAMS + OFF_W1 + (size_t)k * AEV_DIM + n]; break;
        }
        __half hi, lo;
        split_half(v * W_SCALE, hi, lo);
        dst[((size_t)(2 * s) * rows + r) * cols + c] = hi;
        dst[((size_t)(2 * s + 1) * rows + r) * cols + c] = lo;
    }
}
__global__ void k_prep_small(const float* __restrict__ blob, int n_models, float* __restrict__ b1, float* __restrict__ b2,
                             float* __restrict__ b3, float* __restrict__ w4, float* __restrict__ b4) {
    const int s = blockIdx.x;
    for (int e = 0; e < n_models; ++e) {
        const float* net = blob + (size_t)(e * NSP + s) * NET_PARAMS;
        for (int i = threadIdx.x; i < H1; i += blockDim.x) b1[(size_t)s * n_models * H1 + e * H1 + i] = net[OFF_B1 + i];
        for (int i = threadIdx.x; i < H2; i += blockDim.x) b2[(size_t)s * n_models * H2 + e * H2 + i] = net[OFF_B2 + i];
        for (int i = threadIdx.x; i < H3; i += blockDim.x) {
            b3[(size_t)s * n_models * H3 + e * H3 + i] = net[OFF_B3 + i];
            w4[(size_t)s * n_models * H3 + e * H3 + i] = net[OFF_W4 + i];
        }
        if (threadIdx.x == 0) b4[s * n_models + e] = net[OFF_B4];
    }
}

// ---- host ------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
        else
            cudaGetLastError();
    }
    return fn;
}

// 2-D fp16 tensor [rows][cols] row-major, box = 64 columns x box_rows rows, 128-byte swizzle
bool make_map(CUtensorMap* m, const void* ptr, uint64_t rows, uint64_t cols, uint32_t box_rows) {
    EncodeTiledFn enc = get_encode();
    if (!enc) return false;
    cuuint64_t dims[2] = {cols, rows};
    cuuint64_t strides[1] = {cols * 2};
    cuuint32_t box[2] = {BK, box_rows};
    cuuint32_t estr[2] = {1, 1};
    return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, const_cast<void*>(ptr), dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

struct TcWorkspace {                  // per context
    __half* aev;                                   // [2][max_rows][AEV_LD] row-major hi / lo planes (A of G1, via TMA)
    __half *h1, *h2, *d3, *d2, *d1;                // tiled activation planes (see the header); d3 is padded to 192 per model
    int act_models;                                // d1 holds this many networks per row (grown by mlp_tc_ensure)
    int h1_models;                                 // h1 likewise (allocated only where it is an HBM operand); 0 = not allocated
    int lw_models;                                 // h2 / d3 / d2 (layer-by-layer mode only) likewise; 0 = not allocated
    CUtensorMap m_aev;
    __half* fscratch;                              // [SMs][FU_SCRATCH] h1 scratch tiles of k_mlp_fused (L2-resident)
};
struct TcWeights {                    // per weight handle
    __half *w1f, *w2f, *w3f, *w3b, *w2b, *w1b;
    __half* wmid;                                   // k_mlp_mid weight images [species][network][MID_W_TOTAL]
    __half* w1img;                                  // k_mlp_fused W1 images [species][network][64 K steps][FU_W1_STEP]
    float *b1, *b2, *b3, *w4, *b4;
    CUtensorMap m_w1f, m_w2f, m_w3f, m_w3b, m_w2b, m_w1b;
};

template <int EPI, int CMP>
int launch_gemm(Ctx* ctx, const CUtensorMap& a, const CUtensorMap& b, const TcArgs& args) {
    DHP_LAUNCH(ctx, (k_gemm_tc<EPI, CMP>), ctx->sm_count, TC_THREADS, SMEM_BYTES, a, b, args);
    return DHP_OK;
}

template <int EPI, int CMP>
int launch_gemm2(Ctx* ctx, const CUtensorMap& a, const CUtensorMap& b, const TcArgs& args) {
    DHP_LAUNCH(ctx, (k_gemm_tc2<EPI, CMP>), ctx->sm_count, TC_THREADS, T2_SMEM, a, b, args);
    return DHP_OK;
}

}  // namespace

bool mlp_tc_available(Ctx* ctx) { return ctx->cc_major == 10 && get_encode() != nullptr; }

template <int EPI, int CMP>
static int set_smem_tc(Ctx* ctx) {
    DHP_CUDA(ctx, cudaFuncSetAttribute((k_gemm_tc<EPI, CMP>), cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES));
    return DHP_OK;
}

int mlp_tc_alloc(Ctx* ctx) {
    // per-device kernel attributes (dynamic shared memory above 48 KB), once per context
    int rc;
    if ((rc = set_smem_tc<EPI_CELU, CMP_K>(ctx)) != DHP_OK || (rc = set_smem_tc<EPI_CELU, CMP_NONE>(ctx)) != DHP_OK ||
        (rc = set_smem_tc<EPI_OUT, CMP_NONE>(ctx)) != DHP_OK || (rc = set_smem_tc<EPI_DCELU, CMP_NONE>(ctx)) != DHP_OK ||
        (rc = set_smem_tc<EPI_GRAD, CMP_N>(ctx)) != DHP_OK)
        return rc;
    DHP_CUDA(ctx, cudaFuncSetAttribute(k_mlp_mid, cudaFuncAttributeMaxDynamicSharedMemorySize, MID_SMEM));
    DHP_CUDA(ctx, cudaFuncSetAttribute(k_mlp_fused, cudaFuncAttributeMaxDynamicSharedMemorySize, FU_SMEM));
    DHP_CUDA(ctx, cudaFuncSetAttribute((k_gemm_tc2<EPI_CELU, CMP_K>), cudaFuncAttributeMaxDynamicSharedMemorySize, T2_SMEM));
    DHP_CUDA(ctx, cudaFuncSetAttribute((k_gemm_tc2<EPI_GRAD, CMP_N>), cudaFuncAttributeMaxDynamicSharedMemorySize, T2_SMEM));
    TcWorkspace* w = new (std::nothrow) TcWorkspace();
    if (!w) return DHP_E_NOMEM;
    memset((void*)w, 0, sizeof(*w));
    ctx->tc_ws = w;
    const size_t R = (size_t)ctx->max_rows;
    // the activation planes are sized by the ensemble that is actually loaded (mlp_tc_ensure, from dhp_weights_load)
    if (cudaMalloc((void**)&w->aev, 2 * R * AEV_LD * sizeof(__half)) != cudaSuccess) return DHP_E_NOMEM;
    if (cudaMemset(w->aev, 0, 2 * R * AEV_LD * sizeof(__half)) != cudaSuccess) return DHP_E_CUDA;
    if (cudaMalloc((void**)&w->fscratch, (size_t)ctx->sm_count * FU_SCRATCH * sizeof(__half)) != cudaSuccess) return DHP_E_NOMEM;
    if (cudaMemset(w->fscratch, 0, (size_t)ctx->sm_count * FU_SCRATCH * sizeof(__half)) != cudaSuccess) return DHP_E_CUDA;
    if (!make_map(&w->m_aev, w->aev, 2 * R, AEV_LD, BM)) return DHP_E_CUDA;
    ctx->aev_planes = w->aev;
    return DHP_OK;
}

// Setup-time sizing of the activation planes (4 B per element as fp16 hi / lo): h1 and d1 for `n_models` networks per
// row (16 KB per row at 8 networks), and - only if the layer-by-layer comparison mode is in use - h2, d3, d2.  Grows, never
// shrinks; the planes are zeroed so that padding rows stay finite.  Not a hot call: allocates and synchronises.
int mlp_tc_ensure(Ctx* ctx, int n_models, bool layerwise) {
    TcWorkspace* w = (TcWorkspace*)ctx->tc_ws;
    if (!w) return DHP_OK;
    const size_t R = (size_t)ctx->max_rows;
    auto grow = [&](__half** p, size_t width) -> int {
        if (*p) { cudaStreamSynchronize(ctx->stream); cudaFree(*p); *p = nullptr; }
        if (cudaMalloc((void**)p, 2 * R * width * sizeof(__half)) != cudaSuccess) { cudaGetLastError(); return DHP_E_NOMEM; }
        if (cudaMemset(*p, 0, 2 * R * width * sizeof(__half)) != cudaSuccess) return DHP_E_CUDA;
        return DHP_OK;
    };
    int rc;
    if (n_models > w->act_models) {
        if ((rc = grow(&w->d1, (size_t)n_models * H1)) != DHP_OK) { w->act_models = 0; return rc; }
        w->act_models = n_models;
    }
    // h1 is an HBM operand only on the two-launch path (DHP_TC_FUSE=0) and in the layer-by-layer mode: the fused chain kernel
    // keeps it on chip (8 KB per row and 8 networks less: 0.8 GB at 98 000 atoms)
    if ((!ctx->tc_fuse || layerwise) && n_models > w->h1_models) {
        if ((rc = grow(&w->h1, (size_t)n_models * H1)) != DHP_OK) { w->h1_models = 0; return rc; }
        w->h1_models = n_models;
    }
    if (layerwise && n_models > w->lw_models) {
        if ((rc = grow(&w->h2, (size_t)n_models * H2)) != DHP_OK || (rc = grow(&w->d3, (size_t)n_models * H2)) != DHP_OK ||
            (rc = grow(&w->d2, (size_t)n_models * H2)) != DHP_OK) { w->lw_models = 0; return rc; }
        w->lw_models = n_models;
    }
    return DHP_OK;
}

void mlp_tc_free(Ctx* ctx) {
    TcWorkspace* w = (TcWorkspace*)ctx->tc_ws;
    if (!w) return;
    __half* ptrs[] = {w->aev, w->h1, w->h2, w->d3, w->d2, w->d1};
    for (__half* p : ptrs) if (p) cudaFree(p);
    if (w->fscratch) cudaFree(w->fscratch);
    delete w;
    ctx->tc_ws = nullptr;
    ctx->aev_planes = nullptr;
}

int mlp_tc_weights(Ctx* ctx, Weights* wt) {
    TcWeights* t = new (std::nothrow) TcWeights();
    if (!t) return DHP_E_NOMEM;
    memset((void*)t, 0, sizeof(*t));
    wt->tc = t;
    const int M = wt->n_models;
    struct { __half** p; int mode, rows, cols; CUtensorMap* m; uint32_t box_rows; } mats[] = {
        {&t->w1f, WP_W1F, M * H1, AEV_LD, &t->m_w1f, (uint32_t)H1}, {&t->w2f, WP_W2F, M * H2, H1, &t->m_w2f, (uint32_t)H2},
        {&t->w3f, WP_W3F, M * H3, H2, &t->m_w3f, (uint32_t)H3},     {&t->w3b, WP_W3B, M * H2, H3, &t->m_w3b, (uint32_t)H2},
        {&t->w2b, WP_W2B, M * H1, H2, &t->m_w2b, (uint32_t)H1},     {&t->w1b, WP_W1B, AEV_LD, M * H1, &t->m_w1b, (uint32_t)KBLK}};
    for (auto& m : mats) {
        const size_t n = (size_t)2 * NSP * m.rows * m.cols;
        if (cudaMalloc((void**)m.p, n * sizeof(__half)) != cudaSuccess) return DHP_E_NOMEM;
        DHP_LAUNCH(ctx, k_prep_weights, dim3(256, NSP), 256, 0, wt->blob, M, m.mode, m.rows, m.cols, *m.p);
        if (!make_map(m.m, *m.p, (uint64_t)2 * NSP * m.rows, m.cols, m.box_rows)) return DHP_E_CUDA;
    }
    if (cudaMalloc((void**)&t->wmid, (size_t)NSP * M * MID_W_TOTAL * sizeof(__half)) != cudaSuccess) return DHP_E_NOMEM;
    DHP_LAUNCH(ctx, k_prep_mid, dim3(64, NSP * M), 256, 0, wt->blob, M, t->wmid);
    if (cudaMalloc((void**)&t->w1img, (size_t)NSP * M * (AEV_LD / 16) * FU_W1_STEP * sizeof(__half)) != cudaSuccess) return DHP_E_NOMEM;
    DHP_LAUNCH(ctx, k_prep_w1img, dim3(128, NSP * M), 256, 0, wt->blob, M, t->w1img);
    float** smalls[] = {&t->b1, &t->b2, &t->b3, &t->w4, &t->b4};
    const size_t sizes[] = {(size_t)NSP * M * H1, (size_t)NSP * M * H2, (size_t)NSP * M * H3, (size_t)NSP * M * H3, (size_t)NSP * M};
    for (int i = 0; i < 5; ++i)
        if (cudaMalloc((void**)smalls[i], sizes[i] * sizeof(float)) != cudaSuccess) return DHP_E_NOMEM;
    DHP_LAUNCH(ctx, k_prep_small, NSP, 256, 0, wt->blob, M, t->b1, t->b2, t->b3, t->w4, t->b4);
    DHP_CUDA(ctx, cudaGetLastError());
    DHP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return DHP_OK;
}

void mlp_tc_weights_free(Ctx*, Weights* wt) {
    TcWeights* t = (TcWeights*)wt->tc;
    if (!t) return;
    void* ptrs[] = {t->w1f, t->w2f, t->w3f, t->w3b, t->w2b, t->w1b, t->wmid, t->w1img, t->b1, t->b2, t->b3, t->w4, t->b4};
    for (void* p : ptrs) if (p) cudaFree(p);
    delete t;
    wt->tc = nullptr;
}

int mlp_tc(Ctx* ctx, const Weights* wt, bool forward_only) {
    if (ctx->n_atoms == 0) { prof_mark(ctx, DHP_PHASE_MLP_MID); prof_mark(ctx, DHP_PHASE_MLP_B1); return DHP_OK; }
    TcWorkspace* ws = (TcWorkspace*)ctx->tc_ws;
    const TcWeights* t = (const TcWeights*)wt->tc;
    if (!ws || !t) return DHP_E_NOTIMPL;
    const int M = wt->n_models;
    const int R = (int)ctx->max_rows;
    int rc;
    if (M > ws->act_models || (ctx->mlp_mode == DHP_MLP_TENSOR_LAYERWISE && M > ws->lw_models)) return DHP_E_NOTIMPL;   // mlp_tc_ensure not run
    if ((!ctx->tc_fuse || ctx->mlp_mode == DHP_MLP_TENSOR_LAYERWISE) && M > ws->h1_models) return DHP_E_NOTIMPL;
    // e_atom and the tile schedulers were zeroed with the rest of the per-call arena at the start of the call (nlist_build)
    if (!ctx->aev_in_planes)     // rows came from a forward pass in fp32 (debug / mixed use): split them here
        DHP_LAUNCH(ctx, k_split_rows, 4 * ctx->sm_count, 256, 0, ctx->aev, AEV_LD, ctx->sp_start, AEV_LD, ws->aev, R);

    TcArgs a{};
    a.single = ctx->mlp_mode == DHP_MLP_TENSOR_FP16 ? 1 : 0;
    a.row_species = ctx->row_species; a.sp_start = ctx->sp_start; a.alpha = ctx->params.celu_alpha;
    a.inv_models = 1.0f / (float)M; a.a_plane_rows = R; a.plane_tiles = R / BM; a.e_atom = ctx->e_atom;
    a.w4 = t->w4; a.b4 = t->b4; a.tile_mask = ctx->tile_mask;
    const int KB1 = H1 / BK, KB2 = H2 / BK;         // 64-column blocks per model: 4 (h1, d1), 3 (h2, d2, and d3 padded to 192)
    // G1: AEV rows (row-major, TMA) -> h1
    a.K = AEV_LD; a.BN = H1; a.n_tiles = M; a.a_k_off_per_tile = 0; a.b_rows_per_species = M * H1; a.b_rows_per_tile = H1;
    a.acc_scale = 1.0f / W_SCALE; a.bias = t->b1;
    a.a_tiled = ws->aev; a.a_kblocks = N_KBLK; a.a_kb_per_tile = 0;      // the AEV planes are in the tiled operand layout: plain bulk copies
    a.out_planes = ws->h1; a.out_kblocks = M * KB1; a.out_cols_per_tile = H1;
    a.sched = ctx->tc_sched + 0;
    const bool fusedp = ctx->mlp_mode != DHP_MLP_TENSOR_LAYERWISE;
    // two row tiles per CTA (k_gemm_tc2) pay when there are enough tile pairs to keep every SM busy for several items
    const int64_t n_pairs_bound = (ctx->n_atoms + 2 * ROW_TILE - 1) / (2 * ROW_TILE);
    const bool big = n_pairs_bound * M >= 12 * (int64_t)ctx->sm_count;
    const bool two_g1 = fusedp && ((ctx->tc_two & 1) != 0) && big;
    const bool two_b1 = fusedp && ((ctx->tc_two & 2) != 0) && big;
    // G1 fused into the front of the middle chain (k_mlp_fused): no G1 launch, h1 never becomes an HBM operand
    const bool fuse1 = fusedp && ctx->tc_fuse != 0;
    if (fuse1) rc = DHP_OK;
    else if (two_g1) rc = launch_gemm2<EPI_CELU, CMP_K>(ctx, ws->m_aev, t->m_w1f, a);
    else rc = launch_gemm<EPI_CELU, CMP_K>(ctx, ws->m_aev, t->m_w1f, a);
    if (rc != DHP_OK) return rc;
    prof_mark(ctx, DHP_PHASE_MLP_MID);
    if (fuse1) {
        FusedArgs m{};
        m.single = a.single; m.forward_only = forward_only ? 1 : 0; m.n_models = M; m.plane_tiles = R / BM;
        m.row_species = ctx->row_species; m.sp_start = ctx->sp_start; m.tile_mask = ctx->tile_mask;
        m.aev = ws->aev; m.w1img = t->w1img; m.wimg = t->wmid; m.scratch = ws->fscratch; m.d1 = ws->d1;
        m.b1 = t->b1; m.b2 = t->b2; m.b3 = t->b3; m.w4 = t->w4; m.b4 = t->b4;
        m.inv_models = 1.0f / (float)M; m.alpha = ctx->params.celu_alpha; m.e_atom = ctx->e_atom; m.sched = ctx->tc_sched + 1;
        DHP_LAUNCH(ctx, k_mlp_fused, ctx->sm_count, MID_THREADS, FU_SMEM, m);
    } else if (ctx->mlp_mode != DHP_MLP_TENSOR_LAYERWISE) {
        // G2 .. B2 fused: h1 -> d1 with h2, d3, d2 kept on chip
        MidArgs m{};
        m.single = a.single;
        m.row_species = ctx->row_species; m.sp_start = ctx->sp_start; m.n_models = M; m.plane_tiles = R / BM;
        m.h1 = ws->h1; m.d1 = ws->d1; m.wimg = t->wmid; m.b2 = t->b2; m.b3 = t->b3; m.w4 = t->w4; m.b4 = t->b4;
        m.inv_models = 1.0f / (float)M; m.alpha = ctx->params.celu_alpha; m.e_atom = ctx->e_atom; m.sched = ctx->tc_sched + 1;
        m.forward_only = forward_only ? 1 : 0;
        DHP_LAUNCH(ctx, k_mlp_mid, ctx->sm_count, MID_THREADS, MID_SMEM, m);
    } else {
        // G2: h1 -> h2
        a.K = H1; a.BN = H2; a.b_rows_per_species = M * H2; a.b_rows_per_tile = H2; a.bias = t->b2;
        a.a_tiled = ws->h1; a.a_kblocks = M * KB1; a.a_kb_per_tile = KB1;
        a.out_planes = ws->h2; a.out_kblocks = M * KB2; a.out_cols_per_tile = H2;
        a.sched = ctx->tc_sched + 1;
        if ((rc = launch_gemm<EPI_CELU, CMP_NONE>(ctx, ws->m_aev, t->m_w2f, a)) != DHP_OK) return rc;
        // G3 + output layer + seed of the backward pass: h2 -> d3
        a.K = H2; a.BN = H3; a.b_rows_per_species = M * H3; a.b_rows_per_tile = H3; a.bias = t->b3;
        a.a_tiled = ws->h2; a.a_kblocks = M * KB2; a.a_kb_per_tile = KB2;
        a.out_planes = ws->d3; a.out_kblocks = M * KB2; a.out_cols_per_tile = H2;
        a.sched = ctx->tc_sched + 2;
        if ((rc = launch_gemm<EPI_OUT, CMP_NONE>(ctx, ws->m_aev, t->m_w3f, a)) != DHP_OK) return rc;
        if (forward_only) { prof_mark(ctx, DHP_PHASE_MLP_B1); DHP_CUDA(ctx, cudaGetLastError()); return DHP_OK; }
        // B3: d3 -> d2
        a.K = H3; a.BN = H2; a.b_rows_per_species = M * H2; a.b_rows_per_tile = H2;
        a.a_tiled = ws->d3; a.a_kblocks = M * KB2; a.a_kb_per_tile = KB2;
        a.h_planes = ws->h2; a.out_planes = ws->d2; a.out_kblocks = M * KB2; a.out_cols_per_tile = H2;
        a.sched = ctx->tc_sched + 3;
        if ((rc = launch_gemm<EPI_DCELU, CMP_NONE>(ctx, ws->m_aev, t->m_w3b, a)) != DHP_OK) return rc;
        // B2: d2 -> d1
        a.K = H2; a.BN = H1; a.b_rows_per_species = M * H1; a.b_rows_per_tile = H1;
        a.a_tiled = ws->d2; a.a_kblocks = M * KB2; a.a_kb_per_tile = KB2;
        a.h_planes = ws->h1; a.out_planes = ws->d1; a.out_kblocks = M * KB1; a.out_cols_per_tile = H1;
        a.sched = ctx->tc_sched + 4;
        if ((rc = launch_gemm<EPI_DCELU, CMP_NONE>(ctx, ws->m_aev, t->m_w2b, a)) != DHP_OK) return rc;
    }
    prof_mark(ctx, DHP_PHASE_MLP_B1);
    if (forward_only) { DHP_CUDA(ctx, cudaGetLastError()); return DHP_OK; }
    // B1: d1 (all models along K) -> dE/dAEV, only the feature blocks that are active for the row tile
    a.K = M * H1; a.BN = 256; a.n_tiles = AEV_LD / 256; a.b_rows_per_species = AEV_LD; a.b_rows_per_tile = 256;
    a.a_tiled = ws->d1; a.a_kblocks = M * KB1; a.a_kb_per_tile = 0;
    a.acc_scale = 1.0f / (W_SCALE * D_SCALE); a.out_f32 = ctx->grad; a.out_ld = AEV_LD;
    a.sched = ctx->tc_sched + 5;
    {   // small systems: fewer row tiles than SMs -> split K (all networks' 64-wide blocks) over several CTAs per tile
        const int64_t tiles_bound = (ctx->n_atoms + ROW_TILE - 1) / ROW_TILE + 2 * NSP;   // row tiles incl. group padding
        const int KBt = (M * H1) / BK;                                                       // 4 K blocks per network
        int ks = 1;
        while (ks * 2 <= KBt && KBt % (ks * 2) == 0 && tiles_bound * ks * 2 <= ctx->sm_count) ks *= 2;
        a.ksplit = two_b1 ? 1 : ks;
        if (a.ksplit > 1)
            DHP_CUDA(ctx, cudaMemsetAsync(ctx->grad, 0, sizeof(float) * (size_t)std::min<int64_t>(tiles_bound * ROW_TILE, ctx->max_rows) * AEV_LD,
                                          ctx->stream));
    }
    if (two_b1) rc = launch_gemm2<EPI_GRAD, CMP_N>(ctx, ws->m_aev, t->m_w1b, a);
    else rc = launch_gemm<EPI_GRAD, CMP_N>(ctx, ws->m_aev, t->m_w1b, a);
    if (rc != DHP_OK) return rc;
    DHP_CUDA(ctx, cudaGetLastError());
    return DHP_OK;
}

}  // namespace dhp
