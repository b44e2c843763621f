// api.cu -- the C-ABI of libmlp_b200 (include/mlp.h): argument validation, library state,
// lazily created device scratch, host-buffer (end-to-end) entry points.  No arithmetic of the
// method lives here; every step of the path runs in the kernels of the other translation units.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <vector>

#include "../../include/mlp.h"
#include "internal.h"

namespace {

using namespace mlp;

struct State {
    bool init = false;
    uint64_t seed = 0;
    int in = 0, hidden = 0, out = 0;
    int cluster = 0;                  // 0 = automatic
    int num_sms = 0;
    // scratch
    double* eval_partials = nullptr;  int eval_partials_cap = 0;
    double* eval_out = nullptr;       // device double for the synchronous entry
    unsigned long long* stats = nullptr;
    UnfusedScratch unf = {};          int unf_batch = 0, unf_hidden = 0;
    float *priorXT = nullptr, *priorHT = nullptr;   // transposes of the paper's tiled strategy
    float *shufX = nullptr, *shufY = nullptr; size_t shufX_cap = 0, shufY_cap = 0;   // mlp_train_rows
    float *hX = nullptr, *hY = nullptr, *hW1 = nullptr, *hW2 = nullptr; int32_t* hOrder = nullptr;
    size_t hX_cap = 0, hY_cap = 0, hW_cap = 0, hOrder_cap = 0;
    cudaStream_t host_stream = nullptr;
    int64_t launches = 0;
};
State g;
std::mutex g_mu;
thread_local char g_err[512] = "";

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}
int cuda_fail(cudaError_t e, const char* what) {
    return fail(MLP_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}
#define CK(call)                                                \
    do {                                                        \
        cudaError_t e_ = (call);                                \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call);     \
    } while (0)

int ensure_device() {
    if (g.num_sms) return MLP_OK;
    int dev = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&g.num_sms, cudaDevAttrMultiProcessorCount, dev));
    return MLP_OK;
}

template <typename T>
int grow(T** p, size_t* cap, size_t need) {
    if (*cap >= need) return MLP_OK;
    if (*p) CK(cudaFree(*p));
    *p = nullptr; *cap = 0;
    CK(cudaMalloc(reinterpret_cast<void**>(p), need * sizeof(T)));
    *cap = need;
    return MLP_OK;
}

int ensure_eval_scratch(int grid) {
    if (g.eval_partials_cap < grid + 1) {
        if (g.eval_partials) CK(cudaFree(g.eval_partials));
        g.eval_partials = nullptr; g.eval_partials_cap = 0;
        CK(cudaMalloc(reinterpret_cast<void**>(&g.eval_partials), sizeof(double) * (grid + 1)));
        CK(cudaMemset(g.eval_partials, 0, sizeof(double) * (grid + 1)));   // ticket counter = 0
        g.eval_partials_cap = grid + 1;
    }
    if (!g.eval_out) CK(cudaMalloc(reinterpret_cast<void**>(&g.eval_out), sizeof(double)));
    return MLP_OK;
}

int ensure_unfused(int batch, int hidden) {
    if (g.unf.Z1 && g.unf_batch >= batch && g.unf_hidden == hidden) return MLP_OK;
    float** ptrs[] = {&g.unf.Z1, &g.unf.Hact, &g.unf.dZ1, &g.unf.Ypred, &g.unf.dZ2, &g.unf.dW1, &g.unf.dW2,
                      &g.priorXT, &g.priorHT};
    for (auto pp : ptrs) if (*pp) { CK(cudaFree(*pp)); *pp = nullptr; }
    const size_t bh = (size_t)batch * hidden;
    CK(cudaMalloc(reinterpret_cast<void**>(&g.unf.Z1), bh * 4));
    CK(cudaMalloc(reinterpret_cast<void**>(&g.unf.Hact), bh * 4));
    CK(cudaMalloc(reinterpret_cast<void**>(&g.unf.dZ1), bh * 4));
    CK(cudaMalloc(reinterpret_cast<void**>(&g.unf.Ypred), (size_t)batch * 4));
    CK(cudaMalloc(reinterpret_cast<void**>(&g.unf.dZ2), (size_t)batch * 4));
    CK(cudaMalloc(reinterpret_cast<void**>(&g.unf.dW1), (size_t)kIn * hidden * 4));
    CK(cudaMalloc(reinterpret_cast<void**>(&g.unf.dW2), (size_t)hidden * 4));
    CK(cudaMalloc(reinterpret_cast<void**>(&g.priorXT), (size_t)batch * kIn * 4));
    CK(cudaMalloc(reinterpret_cast<void**>(&g.priorHT), bh * 4));
    g.unf_batch = batch; g.unf_hidden = hidden;
    return MLP_OK;
}

int effective_cluster() {
    return g.cluster ? g.cluster : fused_default_cluster(g.hidden);
}

int check_train_args(const float* X, const float* Y, int64_t n, int batch, float lr, int epochs,
                     const float* W1, const float* W2, int variant) {
    if (!g.init) return fail(MLP_ERR_NOT_INIT, "mlp_init has not been called");
    if (!X || !Y || !W1 || !W2) return fail(MLP_ERR_BAD_ARG, "NULL pointer argument");
    if (n < 1) return fail(MLP_ERR_BAD_ARG, "n must be >= 1 (got %lld)", (long long)n);
    if (batch < 1) return fail(MLP_ERR_BAD_ARG, "batch must be >= 1 (got %d)", batch);
    if (epochs < 0) return fail(MLP_ERR_BAD_ARG, "epochs must be >= 0 (got %d)", epochs);
    if (!std::isfinite(lr)) return fail(MLP_ERR_BAD_ARG, "lr must be finite");
    if (variant != MLP_VARIANT_FUSED && variant != MLP_VARIANT_UNFUSED && variant != MLP_VARIANT_TF32 &&
        variant != MLP_VARIANT_PRIOR_NAIVE && variant != MLP_VARIANT_PRIOR_TILED)
        return fail(MLP_ERR_UNSUPPORTED, "training variant %d is not supported", variant);
    if (((uintptr_t)X & 15) || ((uintptr_t)W1 & 15))
        return fail(MLP_ERR_ALIGN, "X and W1 must be 16-byte aligned");
    if (((uintptr_t)Y & 3) || ((uintptr_t)W2 & 3))
        return fail(MLP_ERR_ALIGN, "Y and W2 must be 4-byte aligned");
    const int64_t nb = (n + batch - 1) / batch;
    if (nb > 0x7fffffffLL) return fail(MLP_ERR_BAD_ARG, "too many batches per epoch (batch indices are int32)");
    if (nb * (int64_t)epochs > (int64_t)1 << 40) return fail(MLP_ERR_BAD_ARG, "too many steps");
    return MLP_OK;
}

int train_impl(const float* X, const float* Y, int64_t n, int batch, float lr, int epochs,
               float* W1, float* W2, const int32_t* order, int variant, cudaStream_t stream) {
    int rc = check_train_args(X, Y, n, batch, lr, epochs, W1, W2, variant);
    if (rc) return rc;
    if (epochs == 0) return MLP_OK;
    if ((rc = ensure_device())) return rc;
    if (variant == MLP_VARIANT_FUSED) {
        const int C = effective_cluster();
        if (!fused_supported(g.hidden, C))
            return fail(MLP_ERR_UNSUPPORTED, "cluster %d unsupported for hidden %d", C, g.hidden);
        if (!g.stats) {
            CK(cudaMalloc(reinterpret_cast<void**>(&g.stats), 4 * sizeof(unsigned long long)));
            CK(cudaMemset(g.stats, 0, 4 * sizeof(unsigned long long)));
        }
        cudaError_t e = launch_train_fused(X, Y, n, batch, lr, epochs, W1, W2, order, g.hidden, C,
                                           g.stats, stream, &g.launches);
        if (e != cudaSuccess) return cuda_fail(e, "launch_train_fused");
        return MLP_OK;
    }
    if (variant == MLP_VARIANT_TF32) {
        if (!train_tf32_supported(g.hidden))
            return fail(MLP_ERR_UNSUPPORTED, "TF32 training variant supports hidden 32..256 (got %d)", g.hidden);
        cudaError_t e = launch_train_tf32(X, Y, n, batch, lr, epochs, W1, W2, order, g.hidden, stream, &g.launches);
        if (e != cudaSuccess) return cuda_fail(e, "launch_train_tf32");
        return MLP_OK;
    }
    // unfused baseline: the host loop needs the batch order on the host
    if ((rc = ensure_unfused(batch > n ? (int)n : batch, g.hidden))) return rc;
    std::vector<int32_t> oh;
    if (order) {
        const int64_t nb = (n + batch - 1) / batch;
        oh.resize((size_t)nb * epochs);
        CK(cudaMemcpyAsync(oh.data(), order, oh.size() * 4, cudaMemcpyDeviceToHost, stream));
        CK(cudaStreamSynchronize(stream));
        for (int32_t t : oh)
            if (t < 0 || t >= nb) return fail(MLP_ERR_BAD_ARG, "batch_order entry %d outside [0,%lld)", t, (long long)nb);
    }
    cudaError_t e;
    if (variant == MLP_VARIANT_UNFUSED)
        e = launch_train_unfused(X, Y, n, batch, lr, epochs, W1, W2, order ? oh.data() : nullptr,
                                 g.hidden, g.unf, stream, &g.launches);
    else
        e = launch_train_prior(variant == MLP_VARIANT_PRIOR_TILED, X, Y, n, batch, lr, epochs, W1, W2,
                               order ? oh.data() : nullptr, g.hidden, g.unf, g.priorXT, g.priorHT,
                               stream, &g.launches);
    if (e != cudaSuccess) return cuda_fail(e, "launch_train_unfused/prior");
    return MLP_OK;
}

int eval_impl(const float* X, const float* Y, int64_t n, const float* W1, const float* W2,
              double* d_out, int variant, cudaStream_t stream) {
    if (!g.init) return fail(MLP_ERR_NOT_INIT, "mlp_init has not been called");
    if (!X || !Y || !W1 || !W2 || !d_out) return fail(MLP_ERR_BAD_ARG, "NULL pointer argument");
    if (n < 1) return fail(MLP_ERR_BAD_ARG, "n must be >= 1 (got %lld)", (long long)n);
    if ((uintptr_t)X & 15) return fail(MLP_ERR_ALIGN, "X must be 16-byte aligned");
    int rc = ensure_device();
    if (rc) return rc;
    if (variant == MLP_VARIANT_FUSED) {
        const int grid = eval_fp32_grid(g.hidden, g.num_sms);
        if ((rc = ensure_eval_scratch(grid))) return rc;
        cudaError_t e = launch_eval_fp32(X, Y, n, W1, W2, g.hidden, g.eval_partials, grid, d_out,
                                         stream, &g.launches);
        if (e != cudaSuccess) return cuda_fail(e, "launch_eval_fp32");
        return MLP_OK;
    }
    if (variant == MLP_VARIANT_TF32) {
        if (!eval_tf32_supported(g.hidden))
            return fail(MLP_ERR_UNSUPPORTED, "TF32 eval unsupported for hidden %d", g.hidden);
        const int grid = g.num_sms;
        if ((rc = ensure_eval_scratch(grid))) return rc;
        cudaError_t e = launch_eval_tf32(X, Y, n, W1, W2, g.hidden, g.eval_partials, grid, d_out,
                                         stream, &g.launches);
        if (e != cudaSuccess) return cuda_fail(e, "launch_eval_tf32");
        return MLP_OK;
    }
    return fail(MLP_ERR_UNSUPPORTED, "eval variant %d is not supported", variant);
}

int ensure_host_path(int64_t n, int64_t norder) {
    int rc;
    if ((rc = grow(&g.hX, &g.hX_cap, (size_t)n * kIn))) return rc;
    if ((rc = grow(&g.hY, &g.hY_cap, (size_t)n))) return rc;
    const size_t wn = (size_t)kIn * g.hidden + g.hidden;
    if (g.hW_cap < wn) {
        if (g.hW1) CK(cudaFree(g.hW1));
        g.hW1 = nullptr; g.hW_cap = 0;
        CK(cudaMalloc(reinterpret_cast<void**>(&g.hW1), wn * 4));
        g.hW_cap = wn;
    }
    g.hW2 = g.hW1 + (size_t)kIn * g.hidden;
    if (norder > 0 && (rc = grow(&g.hOrder, &g.hOrder_cap, (size_t)norder))) return rc;
    if (!g.host_stream) CK(cudaStreamCreateWithFlags(&g.host_stream, cudaStreamNonBlocking));
    return MLP_OK;
}

}  // namespace

extern "C" {

int mlp_init(uint64_t seed, int in, int hidden, int out) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (in != 32 || out != 1)
        return fail(MLP_ERR_UNSUPPORTED, "only in=32, out=1 are supported (got in=%d out=%d)", in, out);
    if (hidden != 32 && hidden != 64 && hidden != 128 && hidden != 256 && hidden != 512 && hidden != 1024)
        return fail(MLP_ERR_UNSUPPORTED, "hidden must be one of 32,64,128,256,512,1024 (got %d)", hidden);
    g.init = true; g.seed = seed; g.in = in; g.hidden = hidden; g.out = out;
    if (g.cluster && !fused_supported(hidden, g.cluster)) g.cluster = 0;
    return MLP_OK;
}

int mlp_init_weights(float* W1, float* W2, void* stream) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g.init) return fail(MLP_ERR_NOT_INIT, "mlp_init has not been called");
    if (!W1 || !W2) return fail(MLP_ERR_BAD_ARG, "NULL pointer argument");
    cudaError_t e = launch_init_weights(g.seed, g.hidden, W1, W2, (cudaStream_t)stream, &g.launches);
    if (e != cudaSuccess) return cuda_fail(e, "launch_init_weights");
    return MLP_OK;
}

int mlp_train(const float* X, const float* Y, int64_t n, int batch, float lr, int epochs,
              float* W1, float* W2, void* stream) {
    std::lock_guard<std::mutex> lk(g_mu);
    return train_impl(X, Y, n, batch, lr, epochs, W1, W2, nullptr, MLP_VARIANT_FUSED, (cudaStream_t)stream);
}

int mlp_train_ex(const float* X, const float* Y, int64_t n, int batch, float lr, int epochs,
                 float* W1, float* W2, const int32_t* batch_order, int variant, void* stream) {
    std::lock_guard<std::mutex> lk(g_mu);
    return train_impl(X, Y, n, batch, lr, epochs, W1, W2, batch_order, variant, (cudaStream_t)stream);
}

double mlp_eval_loss(const float* X, const float* Y, int64_t n, const float* W1, const float* W2,
                     void* stream) {
    std::lock_guard<std::mutex> lk(g_mu);
    int rc = ensure_device();
    if (!rc) rc = ensure_eval_scratch(g.num_sms);
    if (rc) return NAN;
    rc = eval_impl(X, Y, n, W1, W2, g.eval_out, MLP_VARIANT_FUSED, (cudaStream_t)stream);
    if (rc) return NAN;
    double h = NAN;
    cudaError_t e = cudaMemcpyAsync(&h, g.eval_out, sizeof(double), cudaMemcpyDeviceToHost, (cudaStream_t)stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize((cudaStream_t)stream);
    if (e != cudaSuccess) { cuda_fail(e, "mlp_eval_loss readback"); return NAN; }
    return h;
}

int mlp_eval_loss_async(const float* X, const float* Y, int64_t n, const float* W1,
                        const float* W2, double* d_out, int variant, void* stream) {
    std::lock_guard<std::mutex> lk(g_mu);
    return eval_impl(X, Y, n, W1, W2, d_out, variant, (cudaStream_t)stream);
}

int mlp_train_rows(const float* X, const float* Y, int64_t n, int batch, float lr, int epochs,
                   float* W1, float* W2, const int32_t* row_order, void* stream) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!row_order) return fail(MLP_ERR_BAD_ARG, "NULL pointer argument");
    int rc = check_train_args(X, Y, n, batch, lr, epochs, W1, W2, MLP_VARIANT_FUSED);
    if (rc) return rc;
    if (n > 0x7fffffffLL / 8) return fail(MLP_ERR_BAD_ARG, "n too large for int32 row indices");
    if ((rc = grow(&g.shufX, &g.shufX_cap, (size_t)n * kIn))) return rc;
    if ((rc = grow(&g.shufY, &g.shufY_cap, (size_t)n))) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    for (int e = 0; e < epochs; ++e) {
        cudaError_t err = launch_gather_rows(X, Y, row_order + (int64_t)e * n, g.shufX, g.shufY, n, st, &g.launches);
        if (err != cudaSuccess) return cuda_fail(err, "launch_gather_rows");
        if ((rc = train_impl(g.shufX, g.shufY, n, batch, lr, 1, W1, W2, nullptr, MLP_VARIANT_FUSED, st))) return rc;
    }
    return MLP_OK;
}

int mlp_train_host(const float* X_host, const float* Y_host, int64_t n, int batch, float lr,
                   int epochs, float* W1_host, float* W2_host, const int32_t* order_host,
                   int variant) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g.init) return fail(MLP_ERR_NOT_INIT, "mlp_init has not been called");
    if (!X_host || !Y_host || !W1_host || !W2_host) return fail(MLP_ERR_BAD_ARG, "NULL pointer argument");
    if (n < 1 || batch < 1 || epochs < 0) return fail(MLP_ERR_BAD_ARG, "bad n/batch/epochs");
    const int64_t nb = (n + batch - 1) / batch;
    const int64_t norder = order_host ? nb * epochs : 0;
    int rc = ensure_host_path(n, norder);
    if (rc) return rc;
    cudaStream_t st = g.host_stream;
    const size_t n1 = (size_t)kIn * g.hidden;
    CK(cudaMemcpyAsync(g.hX, X_host, (size_t)n * kIn * 4, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(g.hY, Y_host, (size_t)n * 4, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(g.hW1, W1_host, n1 * 4, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(g.hW2, W2_host, (size_t)g.hidden * 4, cudaMemcpyHostToDevice, st));
    if (norder) CK(cudaMemcpyAsync(g.hOrder, order_host, (size_t)norder * 4, cudaMemcpyHostToDevice, st));
    rc = train_impl(g.hX, g.hY, n, batch, lr, epochs, g.hW1, g.hW2, norder ? g.hOrder : nullptr, variant, st);
    if (rc) return rc;
    CK(cudaMemcpyAsync(W1_host, g.hW1, n1 * 4, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(W2_host, g.hW2, (size_t)g.hidden * 4, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return MLP_OK;
}

double mlp_eval_loss_host(const float* X_host, const float* Y_host, int64_t n,
                          const float* W1_host, const float* W2_host, int variant) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g.init) { fail(MLP_ERR_NOT_INIT, "mlp_init has not been called"); return NAN; }
    if (!X_host || !Y_host || !W1_host || !W2_host || n < 1) { fail(MLP_ERR_BAD_ARG, "bad argument"); return NAN; }
    if (ensure_host_path(n, 0) || ensure_device() || ensure_eval_scratch(g.num_sms)) return NAN;
    cudaStream_t st = g.host_stream;
    const size_t n1 = (size_t)kIn * g.hidden;
    cudaError_t e = cudaMemcpyAsync(g.hX, X_host, (size_t)n * kIn * 4, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(g.hY, Y_host, (size_t)n * 4, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(g.hW1, W1_host, n1 * 4, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(g.hW2, W2_host, (size_t)g.hidden * 4, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) { cuda_fail(e, "mlp_eval_loss_host H2D"); return NAN; }
    if (eval_impl(g.hX, g.hY, n, g.hW1, g.hW2, g.eval_out, variant, st)) return NAN;
    double h = NAN;
    e = cudaMemcpyAsync(&h, g.eval_out, sizeof(double), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { cuda_fail(e, "mlp_eval_loss_host D2H"); return NAN; }
    return h;
}

int mlp_set_cluster(int cluster) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (cluster == 0) { g.cluster = 0; return MLP_OK; }
    if (!g.init) return fail(MLP_ERR_NOT_INIT, "mlp_init has not been called");
    if (!fused_supported(g.hidden, cluster))
        return fail(MLP_ERR_UNSUPPORTED, "cluster %d unsupported for hidden %d", cluster, g.hidden);
    g.cluster = cluster;
    return MLP_OK;
}

int mlp_get_cluster(void) {
    std::lock_guard<std::mutex> lk(g_mu);
    return g.init ? effective_cluster() : 0;
}

int mlp_get_train_stats(double out[4]) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!out) return fail(MLP_ERR_BAD_ARG, "NULL pointer argument");
    if (!g.stats) return fail(MLP_ERR_NOT_INIT, "no fused training call has run yet");
    unsigned long long h[4];
    CK(cudaMemcpy(h, g.stats, sizeof(h), cudaMemcpyDeviceToHost));
    for (int i = 0; i < 4; ++i) out[i] = (double)h[i];
    return MLP_OK;
}

int64_t mlp_launch_count(void) {
    std::lock_guard<std::mutex> lk(g_mu);
    return g.launches;
}

const char* mlp_last_error(void) { return g_err; }

const char* mlp_version(void) { return "libmlp_b200 0.1 (sm_100a)"; }

void mlp_shutdown(void) {
    std::lock_guard<std::mutex> lk(g_mu);
    void* ptrs[] = {g.eval_partials, g.eval_out, g.stats, g.unf.Z1, g.unf.Hact, g.unf.dZ1,
                    g.unf.Ypred, g.unf.dZ2, g.unf.dW1, g.unf.dW2, g.priorXT, g.priorHT, g.shufX, g.shufY, g.hX, g.hY, g.hW1, g.hOrder};
    for (void* p : ptrs) if (p) cudaFree(p);
    if (g.host_stream) cudaStreamDestroy(g.host_stream);
    const bool init = g.init; const uint64_t seed = g.seed;
    const int in = g.in, hidden = g.hidden, out = g.out, cluster = g.cluster;
    const int64_t launches = g.launches;
    g = State();
    g.init = init; g.seed = seed; g.in = in; g.hidden = hidden; g.out = out; g.cluster = cluster;
    g.launches = launches;
}

}  // extern "C"
