// internal.h -- declarations shared by the translation units of libmlp_b200 (host side).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mlp {

constexpr int kIn = 32;   // input features

// Every launcher returns cudaSuccess or the launch error and adds the kernels it launched
// to *launches.

// train_fused.cu -- persistent fused cluster kernel
// stats: device words [0..3] = SM cycles, ns, steps, cluster; [4] = batch_order entries outside [0, nb)
// (clamped, counted); written by CTA 0 at the end of the launch
bool fused_supported(int hidden, int cluster);
int fused_default_cluster(int hidden, int batch);
cudaError_t launch_train_fused(const float* X, const float* Y, int64_t n, int batch, float lr,
                               int epochs, float* W1, float* W2, const int32_t* order,
                               int hidden, int cluster, unsigned long long* stats,
                               cudaStream_t stream, int64_t* launches);
constexpr int kStatWords = 8;      // words per statistics slot ([5] = row_order entries outside [0, n))

// unfused.cu -- one kernel per equation (row a-U) + weight initialisation
struct UnfusedScratch {
    float *Z1, *Hact, *dZ1;   // [batch x hidden]
    float *Ypred, *dZ2;       // [batch]
    float *dW1, *dW2;         // [32 x hidden], [hidden]
};
cudaError_t launch_train_unfused(const float* X, const float* Y, int64_t n, int batch, float lr,
                                 int epochs, float* W1, float* W2, const int32_t* order_host,
                                 int hidden, const UnfusedScratch& s, cudaStream_t stream,
                                 int64_t* launches);
// prior_art.cu -- the paper's naive / tiled+transposed+fused strategies (comparison only, NEXT-4)
cudaError_t launch_train_prior(bool tiled, const float* X, const float* Y, int64_t n, int batch, float lr,
                               int epochs, float* W1, float* W2, const int32_t* order_host, int hidden,
                               const UnfusedScratch& s, float* XT, float* HT, cudaStream_t stream,
                               int64_t* launches);
cudaError_t launch_gather_rows(const float* X, const float* Y, const int32_t* perm, float* Xp, float* Yp,
                               int64_t n, unsigned long long* bad, cudaStream_t stream, int64_t* launches);
cudaError_t launch_init_weights(uint64_t seed, int hidden, float* W1, float* W2,
                                cudaStream_t stream, int64_t* launches);

// eval_fp32.cu -- streaming forward + MSE (row a-E)
int eval_fp32_grid(int hidden, int num_sms);
cudaError_t launch_eval_fp32(const float* X, const float* Y, int64_t n, const float* W1,
                             const float* W2, int hidden, double* partials, unsigned int* ticket, int grid,
                             double* d_out, cudaStream_t stream, int64_t* launches);

// X viewed as a 2-D tensor [n][32] fp32 with 128-byte swizzle, box = box_rows rows (<= 256); *out_map is a
// CUtensorMap (128 bytes, 64-byte aligned).  False if the driver entry point is unavailable.  atom32: swizzle 32-byte
// chunks (CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B, the layout a TF32 operand needs to be readable MN-major) instead of 16-byte ones.
bool make_x_tensormap(void* out_map, const float* X, int64_t n, int box_rows, bool atom32 = false);

// train_tc.cu -- fused cluster training kernel with eqs. 1 and 8 on the tensor cores (row a-T, separately
// reported): TF32 operands (fp32 bits truncated by the tensor core) or BF16 operands (converted in the kernel,
// round to nearest even), fp32 accumulate, fp32 master weights.
bool train_tc_supported(int hidden, bool bf16);
cudaError_t launch_train_tc(const float* X, const float* Y, int64_t n, int batch, float lr, int epochs,
                            float* W1, float* W2, const int32_t* order, int hidden, bool bf16,
                            unsigned long long* stats, cudaStream_t stream, int64_t* launches);

// eval_tc.cu -- tcgen05 first layer (row a-T, separately reported); variant = MLP_VARIANT_TF32 / _BF16 / _TF32X3
bool eval_tc_supported(int hidden, int variant);
cudaError_t launch_eval_tc(const float* X, const float* Y, int64_t n, const float* W1,
                           const float* W2, int hidden, int variant, double* partials, unsigned int* ticket,
                           int grid, double* d_out, cudaStream_t stream, int64_t* launches);

}  // namespace mlp
