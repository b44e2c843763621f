// api.cu -- the C-ABI of libmlp_b200 (include/mlp.h): argument validation, library state,
// lazily created device scratch, host-buffer (end-to-end) entry points.  No arithmetic of the
// method lives here; every step of the path runs in the kernels of the other translation units.
// (The only sums formed on the host are the fixed-order combination of per-chunk mean losses in
// mlp_eval_loss_host, which is bookkeeping of eq. 4's 1/n, see there.)
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <vector>

#include "../../include/mlp.h"
#include "internal.h"

// Scratch of mlp_eval_loss_static (include/mlp.h): per-CTA partial sums [0, MLP_STATIC_EVAL_MAX_CTAS), then
// the last-block ticket.  File scope, so every GPU that loads this library holds these bytes until exit.  In
// host code this name is only a stand-in for the symbol: the device address comes from cudaGetSymbolAddress
// (static_eval_scratch below), once per device.
constexpr int kStaticEvalDoubles = MLP_STATIC_EVAL_MAX_CTAS + 32;           // 8,448 bytes
static __device__ __align__(256) double g_static_eval_scratch[kStaticEvalDoubles];

namespace {

using namespace mlp;

constexpr int kEvalSlots = 32;     // eval launches in flight that never share a workspace
constexpr int kStatSlots = 64;     // fused training launches in flight with their own statistics
constexpr int kHostChunks = 64;    // at most this many chunks in the pipelined copy of mlp_eval_loss_host
constexpr int64_t kChunkRows = 1 << 18;   // 32 MiB of X per chunk

struct State {
    bool init = false;
    uint64_t seed = 0;
    int in = 0, hidden = 0, out = 0;
    int cluster = 0;                  // 0 = automatic
    int num_sms = 0;
    // Every eval launch gets its own workspace slot (per-CTA partials, ticket, result) and every
    // fused training launch its own statistics slot, so calls on different streams never share
    // library-owned device memory (include/mlp.h, "Concurrency").
    double* eval_pool = nullptr;      // [kEvalSlots][eval_stride]
    size_t eval_stride = 0;           // doubles per slot: num_sms partials + ticket + result
    cudaEvent_t eval_done[kEvalSlots] = {};
    bool eval_zeroed[kEvalSlots] = {};
    unsigned eval_next = 0;
    unsigned long long* stats = nullptr;   // [kStatSlots][kStatWords]
    unsigned stats_next = 0;
    int stats_latest = -1;
    UnfusedScratch unf = {};          int unf_batch = 0, unf_hidden = 0;
    float *priorXT = nullptr, *priorHT = nullptr;   // transposes of the paper's tiled strategy
    float *shufX = nullptr, *shufY = nullptr; size_t shufX_cap = 0, shufY_cap = 0;   // mlp_train_rows
    float *hX = nullptr, *hY = nullptr, *hW1 = nullptr, *hW2 = nullptr; int32_t* hOrder = nullptr;
    double* hLoss = nullptr;
    size_t hX_cap = 0, hY_cap = 0, hW_cap = 0, hOrder_cap = 0, hLoss_cap = 0;
    cudaStream_t host_stream = nullptr, copy_stream = nullptr;
    cudaEvent_t chunk_ev[kHostChunks] = {};
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

// A workspace of the eval kernels: `grid` per-CTA partial sums (double), the last-block ticket, and
// one double for the result of the synchronous entry points.
struct EvalWs {
    double* partials;
    unsigned int* ticket;
    double* result;
    int slot;          // pool slot, or -1 for a caller-supplied workspace
};

size_t eval_ws_doubles() { return (size_t)g.num_sms + 2; }

// Takes the next slot of the pool for a launch on `stream`.  A slot is reused only after the launch
// that last used it has completed: if it has not, `stream` is made to wait for it.  The ticket is
// zeroed on first use, on the launching stream, and re-zeroed by the kernel's last block.
int acquire_eval_slot(cudaStream_t stream, EvalWs* ws) {
    int rc = ensure_device();
    if (rc) return rc;
    if (!g.eval_pool) {
        g.eval_stride = (eval_ws_doubles() + 15) / 16 * 16;       // 128-byte slots
        CK(cudaMalloc(reinterpret_cast<void**>(&g.eval_pool), sizeof(double) * g.eval_stride * kEvalSlots));
        for (int i = 0; i < kEvalSlots; ++i) {
            CK(cudaEventCreateWithFlags(&g.eval_done[i], cudaEventDisableTiming));
            g.eval_zeroed[i] = false;
        }
    }
    const int slot = (int)(g.eval_next++ % kEvalSlots);
    double* base = g.eval_pool + (size_t)slot * g.eval_stride;
    if (!g.eval_zeroed[slot]) {
        CK(cudaMemsetAsync(base, 0, sizeof(double) * g.eval_stride, stream));
        g.eval_zeroed[slot] = true;
    } else if (cudaEventQuery(g.eval_done[slot]) != cudaSuccess) {
        (void)cudaGetLastError();                                  // cudaErrorNotReady is not sticky
        CK(cudaStreamWaitEvent(stream, g.eval_done[slot], 0));
    }
    ws->partials = base;
    ws->ticket = reinterpret_cast<unsigned int*>(base + g.num_sms);
    ws->result = base + g.num_sms + 1;
    ws->slot = slot;
    return MLP_OK;
}

int release_eval_slot(const EvalWs& ws, cudaStream_t stream) {
    if (ws.slot >= 0) CK(cudaEventRecord(g.eval_done[ws.slot], stream));
    return MLP_OK;
}

unsigned long long* acquire_stats_slot() {
    if (!g.stats) {
        if (cudaMalloc(reinterpret_cast<void**>(&g.stats), sizeof(unsigned long long) * kStatWords * kStatSlots) != cudaSuccess ||
            cudaMemset(g.stats, 0, sizeof(unsigned long long) * kStatWords * kStatSlots) != cudaSuccess) {
            g.stats = nullptr;
            return nullptr;
        }
    }
    const int slot = (int)(g.stats_next++ % kStatSlots);
    g.stats_latest = slot;
    return g.stats + (size_t)slot * kStatWords;
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

int effective_cluster(int batch) {
    return g.cluster ? g.cluster : fused_default_cluster(g.hidden, batch);
}

bool known_train_variant(int v) {
    return v == MLP_VARIANT_FUSED || v == MLP_VARIANT_UNFUSED || v == MLP_VARIANT_TF32 || v == MLP_VARIANT_BF16 ||
           v == MLP_VARIANT_PRIOR_NAIVE || v == MLP_VARIANT_PRIOR_TILED;
}

int check_train_args(const float* X, const float* Y, int64_t n, int batch, float lr, int epochs,
                     const float* W1, const float* W2, int variant) {
    if (!g.init) return fail(MLP_ERR_NOT_INIT, "mlp_init has not been called");
    if (!X || !Y || !W1 || !W2) return fail(MLP_ERR_BAD_ARG, "NULL pointer argument");
    if (n < 1) return fail(MLP_ERR_BAD_ARG, "n must be >= 1 (got %lld)", (long long)n);
    if (batch < 1) return fail(MLP_ERR_BAD_ARG, "batch must be >= 1 (got %d)", batch);
    if (epochs < 0) return fail(MLP_ERR_BAD_ARG, "epochs must be >= 0 (got %d)", epochs);
    if (!std::isfinite(lr)) return fail(MLP_ERR_BAD_ARG, "lr must be finite");
    if (!known_train_variant(variant))
        return fail(MLP_ERR_UNSUPPORTED, "training variant %d is not supported", variant);
    if (((uintptr_t)X & 15) || ((uintptr_t)W1 & 15))
        return fail(MLP_ERR_ALIGN, "X and W1 must be 16-byte aligned");
    if (((uintptr_t)Y & 3) || ((uintptr_t)W2 & 3))
        return fail(MLP_ERR_ALIGN, "Y and W2 must be 4-byte aligned");
    const int64_t nb = (n + batch - 1) / batch;
    if (nb > 0x7fffffffLL) return fail(MLP_ERR_BAD_ARG, "too many batches per epoch (batch indices are int32)");
    if (nb * (int64_t)epochs > (int64_t)1 << 40) return fail(MLP_ERR_BAD_ARG, "too many steps");
    const bool per_equation = variant == MLP_VARIANT_UNFUSED || variant == MLP_VARIANT_PRIOR_NAIVE ||
                              variant == MLP_VARIANT_PRIOR_TILED;
    const int64_t rows = batch < n ? batch : n;
    if (per_equation && rows * (int64_t)g.hidden >= (int64_t)1 << 31)
        return fail(MLP_ERR_UNSUPPORTED, "the per-equation baselines index batch x hidden with int32 "
                    "(batch %d x hidden %d is too large)", batch, g.hidden);
    if (per_equation && variant != MLP_VARIANT_UNFUSED && rows > 65535LL * 16)
        return fail(MLP_ERR_UNSUPPORTED, "the paper's 16x16-block kernels put the batch rows in gridDim.y (batch <= 1,048,560)");
    return MLP_OK;
}

// every entry of a host batch-order table must name a batch of the epoch
int check_order_host(const int32_t* order, int64_t count, int64_t nb) {
    for (int64_t k = 0; k < count; ++k)
        if (order[k] < 0 || order[k] >= nb)
            return fail(MLP_ERR_BAD_ARG, "batch_order[%lld] = %d is outside [0, %lld)", (long long)k, order[k],
                        (long long)nb);
    return MLP_OK;
}

int train_impl(const float* X, const float* Y, int64_t n, int batch, float lr, int epochs,
               float* W1, float* W2, const int32_t* order, int variant, cudaStream_t stream,
               unsigned long long* stats_slot = nullptr) {
    int rc = check_train_args(X, Y, n, batch, lr, epochs, W1, W2, variant);
    if (rc) return rc;
    if (epochs == 0) return MLP_OK;
    if ((rc = ensure_device())) return rc;
    if (variant == MLP_VARIANT_FUSED) {
        const int C = effective_cluster(batch);
        if (!fused_supported(g.hidden, C))
            return fail(MLP_ERR_UNSUPPORTED, "cluster %d unsupported for hidden %d", C, g.hidden);
        unsigned long long* st = stats_slot ? stats_slot : acquire_stats_slot();
        if (!st) return cuda_fail(cudaGetLastError(), "statistics slot");
        cudaError_t e = launch_train_fused(X, Y, n, batch, lr, epochs, W1, W2, order, g.hidden, C,
                                           st, stream, &g.launches);
        if (e != cudaSuccess) return cuda_fail(e, "launch_train_fused");
        return MLP_OK;
    }
    if (variant == MLP_VARIANT_TF32 || variant == MLP_VARIANT_BF16) {
        const bool bf16 = variant == MLP_VARIANT_BF16;
        if (!train_tc_supported(g.hidden, bf16))
            return fail(MLP_ERR_UNSUPPORTED, "tensor-core training variant %d does not support hidden %d", variant, g.hidden);
        unsigned long long* st = stats_slot ? stats_slot : acquire_stats_slot();
        if (!st) return cuda_fail(cudaGetLastError(), "statistics slot");
        cudaError_t e = launch_train_tc(X, Y, n, batch, lr, epochs, W1, W2, order, g.hidden, bf16, st, stream, &g.launches);
        if (e != cudaSuccess) return cuda_fail(e, "launch_train_tc");
        return MLP_OK;
    }
    // per-equation baselines: the host loop needs the batch order on the host
    if ((rc = ensure_unfused(batch > n ? (int)n : batch, g.hidden))) return rc;
    std::vector<int32_t> oh;
    if (order) {
        const int64_t nb = (n + batch - 1) / batch;
        oh.resize((size_t)nb * epochs);
        CK(cudaMemcpyAsync(oh.data(), order, oh.size() * 4, cudaMemcpyDeviceToHost, stream));
        CK(cudaStreamSynchronize(stream));
        if ((rc = check_order_host(oh.data(), (int64_t)oh.size(), nb))) return rc;
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

int check_eval_args(const float* X, const float* Y, int64_t n, const float* W1, const float* W2, int variant) {
    if (!g.init) return fail(MLP_ERR_NOT_INIT, "mlp_init has not been called");
    if (!X || !Y || !W1 || !W2) return fail(MLP_ERR_BAD_ARG, "NULL pointer argument");
    if (n < 1) return fail(MLP_ERR_BAD_ARG, "n must be >= 1 (got %lld)", (long long)n);
    if ((uintptr_t)X & 15) return fail(MLP_ERR_ALIGN, "X must be 16-byte aligned");
    if (variant != MLP_VARIANT_FUSED && !eval_tc_supported(g.hidden, variant))
        return fail(MLP_ERR_UNSUPPORTED, "eval variant %d is not supported for hidden %d", variant, g.hidden);
    return MLP_OK;
}

// launches one eval kernel with the given workspace; the mean loss goes to *d_out
int eval_launch(const float* X, const float* Y, int64_t n, const float* W1, const float* W2,
                double* d_out, int variant, const EvalWs& ws, cudaStream_t stream) {
    cudaError_t e;
    if (variant == MLP_VARIANT_FUSED)
        e = launch_eval_fp32(X, Y, n, W1, W2, g.hidden, ws.partials, ws.ticket, eval_fp32_grid(g.hidden, g.num_sms),
                             d_out, stream, &g.launches);
    else
        e = launch_eval_tc(X, Y, n, W1, W2, g.hidden, variant, ws.partials, ws.ticket, g.num_sms, d_out, stream,
                           &g.launches);
    if (e != cudaSuccess) return cuda_fail(e, "eval kernel launch");
    return MLP_OK;
}

// pool-backed eval: the loss goes to *d_out (device); with d_out == nullptr it goes to the slot's own result
// word and is copied to *h_result (host) on the same stream before the slot is released for reuse
int eval_impl(const float* X, const float* Y, int64_t n, const float* W1, const float* W2,
              double* d_out, int variant, cudaStream_t stream, double* h_result = nullptr) {
    int rc = check_eval_args(X, Y, n, W1, W2, variant);
    if (rc) return rc;
    EvalWs ws;
    if ((rc = acquire_eval_slot(stream, &ws))) return rc;
    if (!d_out) d_out = ws.result;
    if ((rc = eval_launch(X, Y, n, W1, W2, d_out, variant, ws, stream))) return rc;
    if (h_result) CK(cudaMemcpyAsync(h_result, ws.result, sizeof(double), cudaMemcpyDeviceToHost, stream));
    return release_eval_slot(ws, stream);
}

int ensure_host_path(int64_t n, int64_t norder, int64_t nloss) {
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
    if (nloss > 0 && (rc = grow(&g.hLoss, &g.hLoss_cap, (size_t)nloss))) return rc;
    if (!g.host_stream) CK(cudaStreamCreateWithFlags(&g.host_stream, cudaStreamNonBlocking));
    if (!g.copy_stream) {
        CK(cudaStreamCreateWithFlags(&g.copy_stream, cudaStreamNonBlocking));
        for (int i = 0; i < kHostChunks; ++i) CK(cudaEventCreateWithFlags(&g.chunk_ev[i], cudaEventDisableTiming));
    }
    return MLP_OK;
}

int check_host_train_args(const float* X_host, const float* Y_host, int64_t n, int batch, int epochs,
                          const float* W1_host, const float* W2_host, const int32_t* order_host) {
    if (!g.init) return fail(MLP_ERR_NOT_INIT, "mlp_init has not been called");
    if (!X_host || !Y_host || !W1_host || !W2_host) return fail(MLP_ERR_BAD_ARG, "NULL pointer argument");
    if (n < 1 || batch < 1 || epochs < 0) return fail(MLP_ERR_BAD_ARG, "bad n/batch/epochs");
    const int64_t nb = (n + batch - 1) / batch;
    if (order_host) return check_order_host(order_host, nb * epochs, nb);      // before anything is copied
    return MLP_OK;
}

// Device address of g_static_eval_scratch and the SM count of the CURRENT device, looked up once per device.
constexpr int kMaxDevices = 64;
double* g_static_ptr[kMaxDevices] = {};
int g_static_sms[kMaxDevices] = {};

int static_eval_scratch(double** ptr, int* sms) {
    int dev = 0;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return fail(MLP_ERR_UNSUPPORTED, "device ordinal %d is outside [0, %d)", dev, kMaxDevices);
    if (!g_static_ptr[dev]) {
        double* p = nullptr;
        CK(cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_static_eval_scratch));
        CK(cudaDeviceGetAttribute(&g_static_sms[dev], cudaDevAttrMultiProcessorCount, dev));
        g_static_ptr[dev] = p;
    }
    *ptr = g_static_ptr[dev];
    *sms = g_static_sms[dev];
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
    double h = NAN;
    {
        std::lock_guard<std::mutex> lk(g_mu);
        if (eval_impl(X, Y, n, W1, W2, nullptr, MLP_VARIANT_FUSED, (cudaStream_t)stream, &h)) return NAN;
    }
    const cudaError_t e = cudaStreamSynchronize((cudaStream_t)stream);
    if (e != cudaSuccess) { cuda_fail(e, "mlp_eval_loss readback"); return NAN; }
    return h;
}

int mlp_eval_loss_async(const float* X, const float* Y, int64_t n, const float* W1,
                        const float* W2, double* d_out, int variant, void* stream) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!d_out) return fail(MLP_ERR_BAD_ARG, "NULL pointer argument");
    return eval_impl(X, Y, n, W1, W2, d_out, variant, (cudaStream_t)stream);
}

size_t mlp_eval_workspace_bytes(void) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (ensure_device()) return 0;
    return sizeof(double) * eval_ws_doubles();
}

int mlp_eval_loss_ws(const float* X, const float* Y, int64_t n, const float* W1, const float* W2,
                     double* d_out, int variant, void* workspace, size_t workspace_bytes, void* stream) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!d_out || !workspace) return fail(MLP_ERR_BAD_ARG, "NULL pointer argument");
    int rc = check_eval_args(X, Y, n, W1, W2, variant);
    if (rc) return rc;
    if ((rc = ensure_device())) return rc;
    if ((uintptr_t)workspace & 7) return fail(MLP_ERR_ALIGN, "workspace must be 8-byte aligned");
    if (workspace_bytes < sizeof(double) * eval_ws_doubles())
        return fail(MLP_ERR_BAD_ARG, "workspace too small: %zu < %zu bytes", workspace_bytes,
                    sizeof(double) * eval_ws_doubles());
    EvalWs ws;
    ws.partials = static_cast<double*>(workspace);
    ws.ticket = reinterpret_cast<unsigned int*>(ws.partials + g.num_sms);
    ws.result = ws.partials + g.num_sms + 1;
    ws.slot = -1;
    return eval_launch(X, Y, n, W1, W2, d_out, variant, ws, (cudaStream_t)stream);
}

int mlp_eval_loss_static(const float* X, const float* Y, int64_t n, const float* W1, const float* W2,
                         double* d_out, int variant, void* stream) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!d_out) return fail(MLP_ERR_BAD_ARG, "NULL pointer argument");
    int rc = check_eval_args(X, Y, n, W1, W2, variant);
    if (rc) return rc;
    double* scratch = nullptr;
    int sms = 0;
    if ((rc = static_eval_scratch(&scratch, &sms))) return rc;
    const int grid = variant == MLP_VARIANT_FUSED ? eval_fp32_grid(g.hidden, sms) : sms;   // one partial sum per CTA
    if (grid > MLP_STATIC_EVAL_MAX_CTAS)
        return fail(MLP_ERR_UNSUPPORTED, "this launch needs %d per-CTA partial sums, the static scratch holds %d "
                    "(MLP_STATIC_EVAL_MAX_CTAS); use mlp_eval_loss_async or mlp_eval_loss_ws", grid,
                    MLP_STATIC_EVAL_MAX_CTAS);
    cudaStream_t st = (cudaStream_t)stream;
    unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch + MLP_STATIC_EVAL_MAX_CTAS);
    // the array keeps what the last call left: the ticket must start at zero, the partial sums are
    // all overwritten before they are read
    CK(cudaMemsetAsync(ticket, 0, sizeof(double), st));
    cudaError_t e;
    if (variant == MLP_VARIANT_FUSED)
        e = launch_eval_fp32(X, Y, n, W1, W2, g.hidden, scratch, ticket, grid, d_out, st, &g.launches);
    else
        e = launch_eval_tc(X, Y, n, W1, W2, g.hidden, variant, scratch, ticket, grid, d_out, st, &g.launches);
    if (e != cudaSuccess) return cuda_fail(e, "eval kernel launch");
    return MLP_OK;
}

int mlp_train_rows(const float* X, const float* Y, int64_t n, int batch, float lr, int epochs,
                   float* W1, float* W2, const int32_t* row_order, void* stream) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!row_order) return fail(MLP_ERR_BAD_ARG, "NULL pointer argument");
    int rc = check_train_args(X, Y, n, batch, lr, epochs, W1, W2, MLP_VARIANT_FUSED);
    if (rc) return rc;
    if (n > 0x7fffffffLL / 8) return fail(MLP_ERR_BAD_ARG, "n too large for int32 row indices");
    if (epochs == 0) return MLP_OK;
    if ((rc = grow(&g.shufX, &g.shufX_cap, (size_t)n * kIn))) return rc;
    if ((rc = grow(&g.shufY, &g.shufY_cap, (size_t)n))) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long* slot = acquire_stats_slot();
    if (!slot) return cuda_fail(cudaGetLastError(), "statistics slot");
    CK(cudaMemsetAsync(slot + 5, 0, sizeof(unsigned long long), st));     // bad row_order entries of this call
    for (int e = 0; e < epochs; ++e) {
        cudaError_t err = launch_gather_rows(X, Y, row_order + (int64_t)e * n, g.shufX, g.shufY, n, slot + 5, st,
                                             &g.launches);
        if (err != cudaSuccess) return cuda_fail(err, "launch_gather_rows");
        if ((rc = train_impl(g.shufX, g.shufY, n, batch, lr, 1, W1, W2, nullptr, MLP_VARIANT_FUSED, st, slot))) return rc;
    }
    return MLP_OK;
}

int mlp_train_host(const float* X_host, const float* Y_host, int64_t n, int batch, float lr,
                   int epochs, float* W1_host, float* W2_host, const int32_t* order_host,
                   int variant) {
    return mlp_fit_host(X_host, Y_host, n, batch, lr, epochs, W1_host, W2_host, order_host, variant,
                        MLP_VARIANT_FUSED, nullptr);
}

int mlp_fit_host(const float* X_host, const float* Y_host, int64_t n, int batch, float lr, int epochs,
                 float* W1_host, float* W2_host, const int32_t* order_host, int variant,
                 int eval_variant, double* epoch_loss_host) {
    std::lock_guard<std::mutex> lk(g_mu);
    int rc = check_host_train_args(X_host, Y_host, n, batch, epochs, W1_host, W2_host, order_host);
    if (rc) return rc;
    const int64_t nb = (n + batch - 1) / batch;
    const int64_t norder = order_host ? nb * epochs : 0;
    if ((rc = ensure_host_path(n, norder, epoch_loss_host ? epochs : 0))) return rc;
    cudaStream_t st = g.host_stream;
    const size_t n1 = (size_t)kIn * g.hidden;
    CK(cudaMemcpyAsync(g.hX, X_host, (size_t)n * kIn * 4, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(g.hY, Y_host, (size_t)n * 4, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(g.hW1, W1_host, n1 * 4, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(g.hW2, W2_host, (size_t)g.hidden * 4, cudaMemcpyHostToDevice, st));
    if (norder) CK(cudaMemcpyAsync(g.hOrder, order_host, (size_t)norder * 4, cudaMemcpyHostToDevice, st));
    if (!epoch_loss_host) {
        // the whole job in one launch (no per-epoch evaluation requested)
        if ((rc = train_impl(g.hX, g.hY, n, batch, lr, epochs, g.hW1, g.hW2, norder ? g.hOrder : nullptr, variant, st)))
            return rc;
    } else {
        // BASELINE.json configs[2]: "a full-dataset eval-loss pass after each epoch": one training launch
        // and one eval launch per epoch, all asynchronous; the losses come back with the weights
        for (int e = 0; e < epochs; ++e) {
            if ((rc = train_impl(g.hX, g.hY, n, batch, lr, 1, g.hW1, g.hW2, norder ? g.hOrder + (int64_t)e * nb : nullptr,
                                 variant, st)))
                return rc;
            if ((rc = eval_impl(g.hX, g.hY, n, g.hW1, g.hW2, g.hLoss + e, eval_variant, st))) return rc;
        }
        if (epochs > 0)
            CK(cudaMemcpyAsync(epoch_loss_host, g.hLoss, sizeof(double) * epochs, cudaMemcpyDeviceToHost, st));
    }
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
    // Pipelined: X/Y go to the device in chunks on a copy stream; the eval kernel of chunk k starts on
    // the compute stream as soon as chunk k has landed, while chunk k+1 is still in flight.  Each
    // chunk's kernel returns the mean over its rows (eq. 4 restricted to the chunk); the dataset loss
    // is the row-weighted mean of those, formed here in chunk order (deterministic).
    int64_t chunk = kChunkRows;
    while ((n + chunk - 1) / chunk > kHostChunks) chunk *= 2;
    const int nchunks = (int)((n + chunk - 1) / chunk);
    if (ensure_host_path(n, 0, nchunks) || ensure_device()) return NAN;
    cudaStream_t st = g.host_stream, cs = g.copy_stream;
    const size_t n1 = (size_t)kIn * g.hidden;
    cudaError_t e = cudaMemcpyAsync(g.hW1, W1_host, n1 * 4, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(g.hW2, W2_host, (size_t)g.hidden * 4, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) { cuda_fail(e, "mlp_eval_loss_host H2D"); return NAN; }
    for (int k = 0; k < nchunks; ++k) {
        const int64_t r0 = (int64_t)k * chunk, rows = (n - r0 < chunk) ? n - r0 : chunk;
        e = cudaMemcpyAsync(g.hX + r0 * kIn, X_host + r0 * kIn, (size_t)rows * kIn * 4, cudaMemcpyHostToDevice, cs);
        if (e == cudaSuccess) e = cudaMemcpyAsync(g.hY + r0, Y_host + r0, (size_t)rows * 4, cudaMemcpyHostToDevice, cs);
        if (e == cudaSuccess) e = cudaEventRecord(g.chunk_ev[k], cs);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(st, g.chunk_ev[k], 0);
        if (e != cudaSuccess) { cuda_fail(e, "mlp_eval_loss_host H2D"); return NAN; }
        if (eval_impl(g.hX + r0 * kIn, g.hY + r0, rows, g.hW1, g.hW2, g.hLoss + k, variant, st)) return NAN;
    }
    std::vector<double> h((size_t)nchunks);
    e = cudaMemcpyAsync(h.data(), g.hLoss, sizeof(double) * nchunks, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(cs);
    if (e != cudaSuccess) { cuda_fail(e, "mlp_eval_loss_host D2H"); return NAN; }
    if (nchunks == 1) return h[0];
    double sse = 0.0;
    for (int k = 0; k < nchunks; ++k) {
        const int64_t r0 = (int64_t)k * chunk, rows = (n - r0 < chunk) ? n - r0 : chunk;
        sse += h[k] * (double)rows;
    }
    return sse / (double)n;
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
    return g.init ? effective_cluster(256) : 0;
}

int mlp_get_cluster_for(int batch) {
    std::lock_guard<std::mutex> lk(g_mu);
    return g.init && batch >= 1 ? effective_cluster(batch) : 0;
}

int mlp_get_train_stats(double out[4]) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!out) return fail(MLP_ERR_BAD_ARG, "NULL pointer argument");
    if (!g.stats || g.stats_latest < 0) return fail(MLP_ERR_NOT_INIT, "no fused training call has run yet");
    unsigned long long h[4];
    CK(cudaMemcpy(h, g.stats + (size_t)g.stats_latest * kStatWords, sizeof(h), cudaMemcpyDeviceToHost));
    for (int i = 0; i < 4; ++i) out[i] = (double)h[i];
    return MLP_OK;
}

int64_t mlp_train_order_errors(void) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g.stats || g.stats_latest < 0) return 0;
    unsigned long long h[2];
    if (cudaMemcpy(h, g.stats + (size_t)g.stats_latest * kStatWords + 4, sizeof(h), cudaMemcpyDeviceToHost) != cudaSuccess) {
        cuda_fail(cudaGetLastError(), "mlp_train_order_errors");
        return -1;
    }
    return (int64_t)(h[0] + h[1]);
}

int64_t mlp_launch_count(void) {
    std::lock_guard<std::mutex> lk(g_mu);
    return g.launches;
}

const char* mlp_last_error(void) { return g_err; }

const char* mlp_version(void) { return "libmlp_b200 0.2 (sm_100a)"; }

void mlp_shutdown(void) {
    std::lock_guard<std::mutex> lk(g_mu);
    void* ptrs[] = {g.eval_pool, g.stats, g.unf.Z1, g.unf.Hact, g.unf.dZ1,
                    g.unf.Ypred, g.unf.dZ2, g.unf.dW1, g.unf.dW2, g.priorXT, g.priorHT, g.shufX, g.shufY, g.hX, g.hY,
                    g.hW1, g.hOrder, g.hLoss};
    for (void* p : ptrs) if (p) cudaFree(p);
    if (g.eval_pool) for (int i = 0; i < kEvalSlots; ++i) if (g.eval_done[i]) cudaEventDestroy(g.eval_done[i]);
    if (g.copy_stream) {
        for (int i = 0; i < kHostChunks; ++i) if (g.chunk_ev[i]) cudaEventDestroy(g.chunk_ev[i]);
        cudaStreamDestroy(g.copy_stream);
    }
    if (g.host_stream) cudaStreamDestroy(g.host_stream);
    const bool init = g.init; const uint64_t seed = g.seed;
    const int in = g.in, hidden = g.hidden, out = g.out, cluster = g.cluster;
    const int64_t launches = g.launches;
    g = State();
    g.init = init; g.seed = seed; g.in = in; g.hidden = hidden; g.out = out; g.cluster = cluster;
    g.launches = launches;
}

}  // extern "C"
