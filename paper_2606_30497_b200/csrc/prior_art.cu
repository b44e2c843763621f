// prior_art.cu -- the paper's own two strategies, re-created from its description for comparison
// only: they are NOT the product path.
//   MLP_VARIANT_PRIOR_NAIVE  "baseline": every product of eqs. 1-8 through one naive matmul kernel,
//       16x16 thread blocks, one thread per output element reading its operands from global
//       memory (eq. 20), ReLU and the other element-wise steps as separate
//       kernels.
//   MLP_VARIANT_PRIOR_TILED  "optimised": 16x16 shared-memory tiles with tile[16][17] padding
//       (PAPER.md:248-258, 375), explicit transposes so both operands are read row-wise
//       (PAPER.md:260-278), ReLU fused into the first product (eq. 23).
// One host-side launch sequence per SGD step, intermediates in HBM -- the structure the paper
// measures.  Every product uses the current weights (reading 16).
#include "common.cuh"
#include "internal.h"

namespace mlp {
namespace {

constexpr int kT = 16;   // TILE_SIZE

// C[M x N] = A' [M x K] * B [K x N];  A' = A (row-major M x K) or, TRANS_A, A stored K x M
template <bool TRANS_A>
__global__ void k_mm_naive(const float* __restrict__ A, const float* __restrict__ B,
                           float* __restrict__ C, int M, int K, int N) {
    const int row = blockIdx.y * kT + threadIdx.y, col = blockIdx.x * kT + threadIdx.x;
    if (row >= M || col >= N) return;
    float sum = 0.f;
    for (int k = 0; k < K; ++k)
        sum = fmaf(TRANS_A ? A[(size_t)k * M + row] : A[(size_t)row * K + k], B[(size_t)k * N + col], sum);
    C[(size_t)row * N + col] = sum;
}

// tiled product, optional fused ReLU
template <bool RELU>
__global__ void k_mm_tiled(const float* __restrict__ A, const float* __restrict__ B,
                           float* __restrict__ C, int M, int K, int N) {
    __shared__ float As[kT][kT + 1], Bs[kT][kT + 1];
    const int row = blockIdx.y * kT + threadIdx.y, col = blockIdx.x * kT + threadIdx.x;
    float sum = 0.f;
    for (int t0 = 0; t0 < K; t0 += kT) {
        const int ka = t0 + threadIdx.x, kb = t0 + threadIdx.y;
        As[threadIdx.y][threadIdx.x] = (row < M && ka < K) ? A[(size_t)row * K + ka] : 0.f;
        Bs[threadIdx.y][threadIdx.x] = (kb < K && col < N) ? B[(size_t)kb * N + col] : 0.f;
        __syncthreads();
#pragma unroll
        for (int k = 0; k < kT; ++k) sum = fmaf(As[threadIdx.y][k], Bs[k][threadIdx.x], sum);
        __syncthreads();
    }
    if (row < M && col < N) C[(size_t)row * N + col] = RELU ? fmaxf(sum, 0.f) : sum;
}

__global__ void k_transpose(const float* __restrict__ in, float* __restrict__ out, int rows, int cols) {
    __shared__ float t[kT][kT + 1];
    int r = blockIdx.y * kT + threadIdx.y, c = blockIdx.x * kT + threadIdx.x;
    if (r < rows && c < cols) t[threadIdx.y][threadIdx.x] = in[(size_t)r * cols + c];
    __syncthreads();
    r = blockIdx.x * kT + threadIdx.y; c = blockIdx.y * kT + threadIdx.x;      // out is cols x rows
    if (r < cols && c < rows) out[(size_t)r * rows + c] = t[threadIdx.x][threadIdx.y];
}

__global__ void k_relu_p(const float* __restrict__ Z, float* __restrict__ Hh, int total) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e < total) Hh[e] = fmaxf(Z[e], 0.f);                                   // eq. 2
}
__global__ void k_dz2_p(const float* __restrict__ Yp, const float* __restrict__ Y, float* __restrict__ d, int m) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < m) d[b] = (2.0f / (float)m) * (Yp[b] - Y[b]);                      // eq. 5
}
// eq. 7: dZ1 = (dZ2 W2^T) (already in dZ1) masked by ReLU'(Z1); H > 0 <=> Z1 > 0
__global__ void k_mask_p(float* __restrict__ dZ1, const float* __restrict__ Hh, int total) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e < total) dZ1[e] = Hh[e] > 0.f ? dZ1[e] : 0.f;
}
__global__ void k_sgd_p(float* __restrict__ W, const float* __restrict__ dW, float lr, int total) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e < total) W[e] = W[e] - lr * dW[e];                                   // eq. 9
}

inline dim3 grid2(int M, int N) { return dim3((N + kT - 1) / kT, (M + kT - 1) / kT); }

}  // namespace

cudaError_t launch_train_prior(bool tiled, const float* X, const float* Y, int64_t n, int batch, float lr,
                               int epochs, float* W1, float* W2, const int32_t* order_host, int hidden,
                               const UnfusedScratch& s, float* XT, float* HT, cudaStream_t stream,
                               int64_t* launches) {
    const int H = hidden;
    const int64_t nb = (n + batch - 1) / batch;
    const dim3 tb(kT, kT);
    for (int e = 0; e < epochs; ++e) {
        for (int64_t k = 0; k < nb; ++k) {
            const int64_t t = order_host ? order_host[(int64_t)e * nb + k] : k;
            const int64_t r0 = t * batch;
            const int m = (int)((n - r0) < batch ? (n - r0) : batch);
            const float* Xb = X + r0 * kIn;
            const float* Yb = Y + r0;
            const int mh = m * H;
            if (!tiled) {
                k_mm_naive<false><<<grid2(m, H), tb, 0, stream>>>(Xb, W1, s.Z1, m, kIn, H);           // eq. 1
                { const cudaError_t e1 = cudaGetLastError(); if (e1 != cudaSuccess) return e1; }
                k_relu_p<<<(mh + 255) / 256, 256, 0, stream>>>(s.Z1, s.Hact, mh);                     // eq. 2
                k_mm_naive<false><<<grid2(m, 1), tb, 0, stream>>>(s.Hact, W2, s.Ypred, m, H, 1);      // eq. 3
                k_dz2_p<<<(m + 255) / 256, 256, 0, stream>>>(s.Ypred, Yb, s.dZ2, m);                  // eq. 5
                k_mm_naive<true><<<grid2(H, 1), tb, 0, stream>>>(s.Hact, s.dZ2, s.dW2, H, m, 1);      // eq. 6
                k_mm_naive<false><<<grid2(m, H), tb, 0, stream>>>(s.dZ2, W2, s.dZ1, m, 1, H);         // eq. 7
                k_mask_p<<<(mh + 255) / 256, 256, 0, stream>>>(s.dZ1, s.Hact, mh);
                k_mm_naive<true><<<grid2(kIn, H), tb, 0, stream>>>(Xb, s.dZ1, s.dW1, kIn, m, H);      // eq. 8
                *launches += 8;
            } else {
                k_mm_tiled<true><<<grid2(m, H), tb, 0, stream>>>(Xb, W1, s.Hact, m, kIn, H);          // eqs. 1-2
                { const cudaError_t e1 = cudaGetLastError(); if (e1 != cudaSuccess) return e1; }
                k_mm_tiled<false><<<grid2(m, 1), tb, 0, stream>>>(s.Hact, W2, s.Ypred, m, H, 1);      // eq. 3
                k_dz2_p<<<(m + 255) / 256, 256, 0, stream>>>(s.Ypred, Yb, s.dZ2, m);                  // eq. 5
                k_transpose<<<grid2(m, H), tb, 0, stream>>>(s.Hact, HT, m, H);
                k_mm_tiled<false><<<grid2(H, 1), tb, 0, stream>>>(HT, s.dZ2, s.dW2, H, m, 1);         // eq. 6
                k_mm_tiled<false><<<grid2(m, H), tb, 0, stream>>>(s.dZ2, W2, s.dZ1, m, 1, H);         // eq. 7
                k_mask_p<<<(mh + 255) / 256, 256, 0, stream>>>(s.dZ1, s.Hact, mh);
                k_transpose<<<grid2(m, kIn), tb, 0, stream>>>(Xb, XT, m, kIn);
                k_mm_tiled<false><<<grid2(kIn, H), tb, 0, stream>>>(XT, s.dZ1, s.dW1, kIn, m, H);     // eq. 8
                *launches += 9;
            }
            k_sgd_p<<<(kIn * H + 255) / 256, 256, 0, stream>>>(W1, s.dW1, lr, kIn * H);               // eq. 9
            k_sgd_p<<<(H + 255) / 256, 256, 0, stream>>>(W2, s.dW2, lr, H);
            *launches += 2;
        }
        cudaError_t err = cudaGetLastError();
        if (err != cudaSuccess) return err;
    }
    return cudaGetLastError();
}

}  // namespace mlp
