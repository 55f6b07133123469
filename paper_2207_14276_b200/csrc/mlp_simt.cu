// a3 + a4 — per-element MLP forward and transpose-backward as fp32 FFMA GEMMs.
//
// This is the small-system path and the numerical scaffold of the tensor path (mlp_tc.cu): plain tiled
// SGEMM, 64x64 tiles, 4x4 register micro-tiles, activations kept in HBM between layers.
// Rows are grouped by the central atom's species (groups start at multiples of ROW_ALIGN = 256 rows), so a
// 64-row tile uses one network; blockIdx.z is the ensemble member.
//   forward : h1 = CELU(G W1^T + b1), h2 = CELU(h1 W2^T + b2), h3 = CELU(h2 W3^T + b3),
//             E_i = (1/M) sum_e (w4 . h3 + b4)
//   backward: d3 = w4 * CELU'(z3) / M, d2 = (d3 W3) * CELU'(z2), d1 = (d2 W2) * CELU'(z1),
//             dE/dG = sum_e d1_e W1_e      (no weight gradients)
// CELU'(z) is recovered from h = CELU(z): 1 if h > 0 else h/alpha + 1.
#include "dhp_internal.cuh"

namespace dhp {

constexpr int TM = 64, TN = 64, TK = 16;

enum { EPI_CELU = 0, EPI_DCELU = 1, EPI_SUM = 2 };

struct GemmArgs {
    const float* A; int lda; int a_model_stride;    // A[row*lda + e*a_model_stride + k]
    const float* W; int w_off;                      // network (e,s) at W + (e*NSP+s)*NET_PARAMS + w_off
    int sbn, sbk;                                   // B(n,k) = Wnet[n*sbn + k*sbk]
    int bias_off;                                   // EPI_CELU
    const float* Hs; int ldh; int h_model_stride;   // EPI_DCELU: saved activations
    float* C; int ldc; int c_model_stride;
    int N, K;
    int n_models;                                   // EPI_SUM: models folded into the K loop
    float alpha;
    const int* kmap;                                // internal AEV column -> canonical feature for the k index (layer 1), or null
    const int* nmap;                                // the same for the n index (dE/dAEV), or null
};

template <int EPI, bool B_KMAJOR>
__global__ void __launch_bounds__(256) k_sgemm(const GemmArgs a, const int* __restrict__ row_species,
                                               const int* __restrict__ sp_start) {
    const int row0 = blockIdx.x * TM;
    if (row0 >= sp_start[NSP]) return;
    const int s = row_species[row0];
    if (s < 0) return;                       // tile made of padding rows only
    const int n0 = blockIdx.y * TN;
    __shared__ float As[TK][TM + 4];
    __shared__ float Bs[TK][TN + 4];
    const int tid = threadIdx.x;
    const int tx = tid & 15, ty = tid >> 4;  // micro-tile: rows ty*4.., cols tx*4..
    float acc[4][4] = {};
    const int e_first = (EPI == EPI_SUM) ? 0 : blockIdx.z;
    const int e_last = (EPI == EPI_SUM) ? a.n_models : blockIdx.z + 1;
    for (int e = e_first; e < e_last; ++e) {
        const float* Ap = a.A + (size_t)row0 * a.lda + (size_t)e * a.a_model_stride;
        const float* Bp = a.W + (size_t)(e * NSP + s) * NET_PARAMS + a.w_off;
        for (int k0 = 0; k0 < a.K; k0 += TK) {
            {   // A tile: 64 rows x 16 k, k contiguous
                int r = tid >> 2, kq = (tid & 3) * 4;
                const float4 v = *reinterpret_cast<const float4*>(Ap + (size_t)r * a.lda + k0 + kq);
                As[kq + 0][r] = v.x; As[kq + 1][r] = v.y; As[kq + 2][r] = v.z; As[kq + 3][r] = v.w;
            }
            if (B_KMAJOR) {
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    int nn = (tid >> 4) + 16 * q, kk = tid & 15;
                    int ng = n0 + nn;
                    const int kf = a.kmap ? a.kmap[k0 + kk] : k0 + kk;
                    Bs[kk][nn] = ng < a.N ? Bp[(size_t)ng * a.sbn + (size_t)kf * a.sbk] : 0.f;
                }
            } else {
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    int nn = tid & 63, kk = (tid >> 6) + 4 * q;
                    int ng = n0 + nn;
                    const int nf = (a.nmap && ng < a.N) ? a.nmap[ng] : ng;
                    Bs[kk][nn] = ng < a.N ? Bp[(size_t)nf * a.sbn + (size_t)(k0 + kk) * a.sbk] : 0.f;
                }
            }
            __syncthreads();
#pragma unroll
            for (int kk = 0; kk < TK; ++kk) {
                const float4 av = *reinterpret_cast<const float4*>(&As[kk][ty * 4]);
                const float4 bv = *reinterpret_cast<const float4*>(&Bs[kk][tx * 4]);
                const float ar[4] = {av.x, av.y, av.z, av.w}, br[4] = {bv.x, bv.y, bv.z, bv.w};
#pragma unroll
                for (int r = 0; r < 4; ++r)
#pragma unroll
                    for (int c = 0; c < 4; ++c) acc[r][c] = fmaf(ar[r], br[c], acc[r][c]);
            }
            __syncthreads();
        }
    }
    const int e = (EPI == EPI_SUM) ? 0 : blockIdx.z;
    const float* bias = a.W + (size_t)(e * NSP + s) * NET_PARAMS + a.bias_off;
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int row = row0 + ty * 4 + r;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int nn = n0 + tx * 4 + c;
            if (nn >= a.N) continue;
            float v = acc[r][c];
            if (EPI == EPI_CELU) {
                v += bias[nn];
                v = v > 0.f ? v : a.alpha * expm1f(v / a.alpha);
            } else if (EPI == EPI_DCELU) {
                float h = a.Hs[(size_t)row * a.ldh + (size_t)e * a.h_model_stride + nn];
                v *= h > 0.f ? 1.0f : h / a.alpha + 1.0f;
            }
            a.C[(size_t)row * a.ldc + (size_t)e * a.c_model_stride + nn] = v;
        }
    }
}

// output layer 160 -> 1 and the seed of the backward pass; one warp per row
__global__ void k_out_layer(const float* __restrict__ h3, const float* __restrict__ W, const int* __restrict__ row_species,
                            const int* __restrict__ sp_start, int n_models, float alpha, float* __restrict__ d3,
                            float* __restrict__ e_atom) {
    const int row = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (row >= sp_start[NSP]) return;
    const int s = row_species[row];
    if (s < 0) return;
    const float inv_m = 1.0f / (float)n_models;
    float esum = 0.f;
    for (int e = 0; e < n_models; ++e) {
        const float* net = W + (size_t)(e * NSP + s) * NET_PARAMS;
        const float* h = h3 + (size_t)row * (n_models * H3) + e * H3;
        float* d = d3 + (size_t)row * (n_models * H3) + e * H3;
        float acc = 0.f;
        for (int k = lane; k < H3; k += 32) {
            float hv = h[k], wv = net[OFF_W4 + k];
            acc = fmaf(wv, hv, acc);
            d[k] = wv * (hv > 0.f ? 1.0f : hv / alpha + 1.0f) * inv_m;
        }
        for (int o = 16; o; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        esum += acc + net[OFF_B4];
    }
    if (lane == 0) e_atom[row] = esum * inv_m;
}

// The fp32 scaffold keeps every activation in HBM (39 KB per row at 8 networks): its buffers exist only once the SIMT path is
// actually going to run, sized by the ensemble in use (setup time, or the first SIMT call).  Grows, never shrinks.
int mlp_simt_ensure(Ctx* ctx, int n_models) {
    if (n_models <= ctx->simt_models) return DHP_OK;
    const size_t R = (size_t)ctx->max_rows;
    const size_t widths[6] = {H1, H2, H3, H3, H2, H1};   // h1 h2 h3 d3 d2 d1
    cudaStreamSynchronize(ctx->stream);
    for (int b = 0; b < 6; ++b) {
        if (ctx->act[b]) { cudaFree(ctx->act[b]); ctx->act[b] = nullptr; }
        if (cudaMalloc(&ctx->act[b], sizeof(float) * R * n_models * widths[b]) != cudaSuccess) { cudaGetLastError(); ctx->simt_models = 0; return DHP_E_NOMEM; }
    }
    ctx->simt_models = n_models;
    return DHP_OK;
}
void mlp_simt_free(Ctx* ctx) {
    for (int b = 0; b < 6; ++b) if (ctx->act[b]) cudaFree(ctx->act[b]);
}

int mlp_simt(Ctx* ctx, const Weights* w, bool forward_only) {
    if (ctx->n_atoms == 0) return DHP_OK;
    const int M = w->n_models;
    const int row_tiles = (int)((ctx->n_atoms + NSP * (ROW_ALIGN - 1) + TM - 1) / TM);   // bound on sp_start[7]/TM
    float *h1 = ctx->act[0], *h2 = ctx->act[1], *h3 = ctx->act[2], *d3 = ctx->act[3], *d2 = ctx->act[4], *d1 = ctx->act[5];
    const float alpha = ctx->params.celu_alpha;
    GemmArgs g{};
    g.W = w->blob; g.alpha = alpha; g.n_models = M;
    // forward
    g.A = ctx->aev; g.lda = AEV_LD; g.a_model_stride = 0; g.w_off = OFF_W1; g.sbn = AEV_DIM; g.sbk = 1; g.bias_off = OFF_B1;
    g.kmap = ctx->col2feat;
    g.C = h1; g.ldc = M * H1; g.c_model_stride = H1; g.N = H1; g.K = AEV_DIM;
    DHP_LAUNCH(ctx, (k_sgemm<EPI_CELU, true>), dim3(row_tiles, H1 / TN, M), 256, 0, g, ctx->row_species, ctx->sp_start);
    g.kmap = nullptr;
    g.A = h1; g.lda = M * H1; g.a_model_stride = H1; g.w_off = OFF_W2; g.sbn = H1; g.bias_off = OFF_B2;
    g.C = h2; g.ldc = M * H2; g.c_model_stride = H2; g.N = H2; g.K = H1;
    DHP_LAUNCH(ctx, (k_sgemm<EPI_CELU, true>), dim3(row_tiles, H2 / TN, M), 256, 0, g, ctx->row_species, ctx->sp_start);
    g.A = h2; g.lda = M * H2; g.a_model_stride = H2; g.w_off = OFF_W3; g.sbn = H2; g.bias_off = OFF_B3;
    g.C = h3; g.ldc = M * H3; g.c_model_stride = H3; g.N = H3; g.K = H2;
    DHP_LAUNCH(ctx, (k_sgemm<EPI_CELU, true>), dim3(row_tiles, (H3 + TN - 1) / TN, M), 256, 0, g, ctx->row_species, ctx->sp_start);
    const int64_t rows_bound = (int64_t)row_tiles * TM;
    DHP_LAUNCH(ctx, k_out_layer, (int)((rows_bound * 32 + 255) / 256), 256, 0, h3, w->blob, ctx->row_species, ctx->sp_start, M,
               alpha, d3, ctx->e_atom);
    if (forward_only) { DHP_CUDA(ctx, cudaGetLastError()); return DHP_OK; }
    // backward: B(n,k) = W[k][n]
    g.A = d3; g.lda = M * H3; g.a_model_stride = H3; g.w_off = OFF_W3; g.sbn = 1; g.sbk = H2;
    g.Hs = h2; g.ldh = M * H2; g.h_model_stride = H2; g.C = d2; g.ldc = M * H2; g.c_model_stride = H2; g.N = H2; g.K = H3;
    DHP_LAUNCH(ctx, (k_sgemm<EPI_DCELU, false>), dim3(row_tiles, H2 / TN, M), 256, 0, g, ctx->row_species, ctx->sp_start);
    g.A = d2; g.lda = M * H2; g.a_model_stride = H2; g.w_off = OFF_W2; g.sbn = 1; g.sbk = H1;
    g.Hs = h1; g.ldh = M * H1; g.h_model_stride = H1; g.C = d1; g.ldc = M * H1; g.c_model_stride = H1; g.N = H1; g.K = H2;
    DHP_LAUNCH(ctx, (k_sgemm<EPI_DCELU, false>), dim3(row_tiles, H1 / TN, M), 256, 0, g, ctx->row_species, ctx->sp_start);
    g.A = d1; g.lda = M * H1; g.a_model_stride = H1; g.w_off = OFF_W1; g.sbn = 1; g.sbk = AEV_DIM;
    g.C = ctx->grad; g.ldc = AEV_LD; g.c_model_stride = 0; g.N = AEV_DIM; g.K = H1; g.nmap = ctx->col2feat;
    DHP_LAUNCH(ctx, (k_sgemm<EPI_SUM, false>), dim3(row_tiles, (AEV_DIM + TN - 1) / TN, 1), 256, 0, g, ctx->row_species, ctx->sp_start);
    DHP_CUDA(ctx, cudaGetLastError());
    return DHP_OK;
}

}  // namespace dhp
