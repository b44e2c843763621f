// unfused.cu -- our own unfused baseline (SURVEY.md 8(a) row a-U): one plain global-memory
// kernel per equation of, launched per SGD step from a host loop, with Z1 / H /
// dZ1 round-tripping through HBM.  This is the structure the paper criticises
// (PAPER.md:162-164, 233-236); it exists for comparison only.  Also: weight initialisation.
#include "common.cuh"
#include "internal.h"

namespace mlp {
namespace {

// eq. 1: Z1[b][j] = sum_i X[b][i] W1[i][j]          one thread per output element
__global__ void k_fwd1(const float* __restrict__ X, const float* __restrict__ W1,
                       float* __restrict__ Z1, int m, int H) {
    int j = blockIdx.y * blockDim.x + threadIdx.x;   // rows in gridDim.x (no 65,535 limit)
    int b = blockIdx.x;
    if (j >= H || b >= m) return;
    float s = 0.f;
    for (int i = 0; i < kIn; ++i) s = fmaf(X[(size_t)b * kIn + i], W1[(size_t)i * H + j], s);
    Z1[(size_t)b * H + j] = s;
}
// eq. 2: H = max(0, Z1)
__global__ void k_relu(const float* __restrict__ Z1, float* __restrict__ Hact, int total) {
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e < total) Hact[e] = fmaxf(Z1[e], 0.f);
}
// eq. 3: Ypred[b] = sum_j H[b][j] W2[j]              one warp per sample, fixed shuffle tree
__global__ void k_fwd2(const float* __restrict__ Hact, const float* __restrict__ W2,
                       float* __restrict__ Ypred, int m, int H) {
    int b = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    int lane = threadIdx.x & 31;
    if (b >= m) return;
    float s = 0.f;
    for (int j = lane; j < H; j += 32) s = fmaf(Hact[(size_t)b * H + j], W2[j], s);
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) Ypred[b] = s;
}
// eq. 5: dZ2 = (2/m)(Ypred - Y)
__global__ void k_dz2(const float* __restrict__ Ypred, const float* __restrict__ Y,
                      float* __restrict__ dZ2, int m) {
    int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < m) dZ2[b] = (2.0f / (float)m) * (Ypred[b] - Y[b]);
}
// eq. 6: dW2[j] = sum_b H[b][j] dZ2[b]               one thread per hidden unit
__global__ void k_dw2(const float* __restrict__ Hact, const float* __restrict__ dZ2,
                      float* __restrict__ dW2, int m, int H) {
    int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= H) return;
    float s = 0.f;
    for (int b = 0; b < m; ++b) s = fmaf(Hact[(size_t)b * H + j], dZ2[b], s);
    dW2[j] = s;
}
// eq. 7: dZ1[b][j] = Z1[b][j] > 0 ? dZ2[b] W2[j] : 0   (W2 not yet updated)
__global__ void k_dz1(const float* __restrict__ Z1, const float* __restrict__ dZ2,
                      const float* __restrict__ W2, float* __restrict__ dZ1, int m, int H) {
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= m * H) return;
    int b = e / H, j = e - b * H;
    dZ1[e] = Z1[e] > 0.f ? dZ2[b] * W2[j] : 0.f;
}
// eq. 8: dW1[i][j] = sum_b X[b][i] dZ1[b][j]         one thread per weight
__global__ void k_dw1(const float* __restrict__ X, const float* __restrict__ dZ1,
                      float* __restrict__ dW1, int m, int H) {
    int j = blockIdx.x * blockDim.x + threadIdx.x;
    int i = blockIdx.y;
    if (j >= H) return;
    float s = 0.f;
    for (int b = 0; b < m; ++b) s = fmaf(X[(size_t)b * kIn + i], dZ1[(size_t)b * H + j], s);
    dW1[(size_t)i * H + j] = s;
}
// eq. 9: W <- W - lr dW for both matrices
__global__ void k_sgd(float* __restrict__ W1, float* __restrict__ W2,
                      const float* __restrict__ dW1, const float* __restrict__ dW2, float lr,
                      int n1, int n2) {
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e < n1) W1[e] = W1[e] - lr * dW1[e];
    else if (e < n1 + n2) W2[e - n1] = W2[e - n1] - lr * dW2[e - n1];
}

// mlp_init_weights: counter-based U(+-1/sqrt(fan_in)), specified in include/mlp.h
__global__ void k_init_weights(unsigned long long seed, int H, float* __restrict__ W1,
                               float* __restrict__ W2) {
    unsigned long long e = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long n1 = (unsigned long long)kIn * H;
    if (e >= n1 + H) return;
    unsigned long long z = seed + 0x9E3779B97F4A7C15ULL * (e + 1);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    z = z ^ (z >> 31);
    double u = (double)(z >> 40) * (1.0 / 16777216.0);
    double bound = 1.0 / sqrt(e < n1 ? (double)kIn : (double)H);
    float w = (float)((2.0 * u - 1.0) * bound);
    if (e < n1) W1[e] = w; else W2[e - n1] = w;
}

// sample-level shuffling: Xp[r] = X[perm[r]], Yp[r] = Y[perm[r]]; one
// float4 per thread, eight threads per 128-byte row
__global__ void k_gather_rows(const float* __restrict__ X, const float* __restrict__ Y,
                              const int* __restrict__ perm, float* __restrict__ Xp,
                              float* __restrict__ Yp, long long n, unsigned long long* __restrict__ bad) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long r = e >> 3;
    if (r >= n) return;
    const int c = (int)(e & 7);
    long long src = perm[r];
    if (src < 0 || src >= n) {                      // row_order entry outside [0, n): clamped, counted, reported
        if (c == 0) atomicAdd(bad, 1ull);
        src = src < 0 ? 0 : n - 1;
    }
    reinterpret_cast<float4*>(Xp)[e] = __ldg(reinterpret_cast<const float4*>(X) + src * 8 + c);
    if (c == 0) Yp[r] = __ldg(Y + src);
}

}  // namespace

cudaError_t launch_gather_rows(const float* X, const float* Y, const int32_t* perm, float* Xp, float* Yp,
                               int64_t n, unsigned long long* bad, cudaStream_t stream, int64_t* launches) {
    const long long total = (long long)n * 8;
    k_gather_rows<<<(unsigned)((total + 255) / 256), 256, 0, stream>>>(X, Y, perm, Xp, Yp, n, bad);
    ++*launches;
    return cudaGetLastError();
}

cudaError_t launch_init_weights(uint64_t seed, int hidden, float* W1, float* W2,
                                cudaStream_t stream, int64_t* launches) {
    int total = kIn * hidden + hidden;
    k_init_weights<<<(total + 255) / 256, 256, 0, stream>>>(seed, hidden, W1, W2);
    ++*launches;
    return cudaGetLastError();
}

cudaError_t launch_train_unfused(const float* X, const float* Y, int64_t n, int batch, float lr,
                                 int epochs, float* W1, float* W2, const int32_t* order_host,
                                 int hidden, const UnfusedScratch& s, cudaStream_t stream,
                                 int64_t* launches) {
    const int H = hidden;
    const int64_t nb = (n + batch - 1) / batch;
    const int tj = H < 128 ? H : 128;
    for (int e = 0; e < epochs; ++e) {
        for (int64_t k = 0; k < nb; ++k) {
            const int64_t t = order_host ? order_host[(int64_t)e * nb + k] : k;
            const int64_t r0 = t * batch;
            const int m = (int)((n - r0) < batch ? (n - r0) : batch);
            const float* Xb = X + r0 * kIn;
            const float* Yb = Y + r0;
            k_fwd1<<<dim3(m, (H + tj - 1) / tj), tj, 0, stream>>>(Xb, W1, s.Z1, m, H);
            {   // a failed first launch must not let the rest of the step run on stale intermediates
                const cudaError_t e1 = cudaGetLastError();
                if (e1 != cudaSuccess) return e1;
            }
            k_relu<<<(m * H + 255) / 256, 256, 0, stream>>>(s.Z1, s.Hact, m * H);
            k_fwd2<<<(m + 7) / 8, 256, 0, stream>>>(s.Hact, W2, s.Ypred, m, H);
            k_dz2<<<(m + 255) / 256, 256, 0, stream>>>(s.Ypred, Yb, s.dZ2, m);
            k_dw2<<<(H + tj - 1) / tj, tj, 0, stream>>>(s.Hact, s.dZ2, s.dW2, m, H);
            k_dz1<<<(m * H + 255) / 256, 256, 0, stream>>>(s.Z1, s.dZ2, W2, s.dZ1, m, H);
            k_dw1<<<dim3((H + tj - 1) / tj, kIn), tj, 0, stream>>>(Xb, s.dZ1, s.dW1, m, H);
            k_sgd<<<(kIn * H + H + 255) / 256, 256, 0, stream>>>(W1, W2, s.dW1, s.dW2, lr,
                                                                 kIn * H, H);
            *launches += 8;
        }
        cudaError_t err = cudaGetLastError();
        if (err != cudaSuccess) return err;
    }
    return cudaGetLastError();
}

}  // namespace mlp
