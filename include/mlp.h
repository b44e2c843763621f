/*
 * mlp.h -- C-ABI of the B200 (sm_100a) mini-batch SGD library for the shallow ReLU/MSE MLP
 * of arxiv/paper_2606_30497 (32-H-1, no bias).
 *
 * What the library computes, per mini-batch of m rows (eqs. 1-9):
 *   (1) Z1 = X W1   (2) H = ReLU(Z1)   (3) Ypred = H W2   (4) L = (1/m) sum (Ypred - Y)^2
 *   (5) dZ2 = (2/m)(Ypred - Y)   (6) dW2 = H^T dZ2   (7) dZ1 = (dZ2 W2^T) (.) [Z1 > 0]
 *   (8) dW1 = X^T dZ1            (9) W <- W - lr dW   (both matrices, after both gradients)
 * iterated over every batch of every epoch.  ReLU'(x) = 1 if x > 0,
 * otherwise 0.  m is the row count of the current batch (a short tail batch
 * uses its own m).  Batches are contiguous row ranges [t*batch, min(n,(t+1)*batch)).
 *
 * Conventions
 *   - Pointers named X, Y, W1, W2, batch_order, d_out are DEVICE pointers owned by the caller
 *     (e.g. torch allocations); pointers with an `_host` suffix are HOST pointers.  The library
 *     never frees or retains caller memory.  Library-owned scratch is created lazily and
 *     released by mlp_shutdown() (mlp_eval_loss_static allocates nothing, see there).
 *   - Layout: all tensors fp32, row-major, dense: X [n x 32], Y [n], W1 [32 x hidden],
 *     W2 [hidden].  X must be 16-byte aligned, Y 4-byte aligned, W1 16-byte aligned.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - Functions returning int return MLP_OK (0) or a positive mlp_status; nothing throws or
 *     calls exit().  Errors detected before launch leave W1/W2 untouched.  mlp_last_error()
 *     describes the most recent failure on the calling thread.
 *   - Concurrency: one model descriptor per process (set by mlp_init).  Calls on different streams
 *     with different caller buffers may overlap on the device: every eval launch takes its own
 *     workspace (per-CTA partial sums, ticket, result) from a library-owned pool of 32 slots, a slot
 *     being reused only after the launch that last used it has completed (the later stream is made
 *     to wait otherwise), and every fused training launch writes its statistics to its own slot
 *     (64 slots).  mlp_eval_loss_ws takes a caller-owned workspace instead; mlp_eval_loss_static
 *     uses ONE file-scope device array for all its calls, which therefore must not overlap on the
 *     device (see there).  The entry points
 *     themselves are serialised by a mutex (enqueueing is cheap; the kernels run asynchronously).
 *   - There is no CPU fallback: without a CUDA device every compute entry returns MLP_ERR_CUDA.
 */
#ifndef PAPER_2606_30497_MLP_H
#define PAPER_2606_30497_MLP_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    MLP_OK = 0,
    MLP_ERR_NOT_INIT = 1,     /* mlp_init has not been called */
    MLP_ERR_BAD_ARG = 2,      /* NULL pointer, n < 1, batch < 1, epochs < 0, non-finite lr, ... */
    MLP_ERR_UNSUPPORTED = 3,  /* dimensions / variant / cluster size outside the supported set */
    MLP_ERR_ALIGN = 4,        /* X or W1 not 16-byte aligned */
    MLP_ERR_CUDA = 5          /* a CUDA runtime call failed (see mlp_last_error) */
} mlp_status;

/* `variant` of mlp_train_ex / mlp_eval_loss_async */
enum {
    MLP_VARIANT_FUSED = 0,    /* training: persistent fused cluster kernel, exact fp32 (FFMA)   */
                              /* eval:     streaming fp32 kernel (FFMA)                          */
    MLP_VARIANT_UNFUSED = 1,  /* training: one kernel per equation, launched per step (baseline) */
    MLP_VARIANT_TF32 = 2,     /* eval: eq. 1, training: eqs. 1 and 8 on the tensor cores (tcgen05.mma kind::tf32: fp32
                                 operands truncated to TF32, fp32 accumulate, fp32 master weights); separately
                                 reported, own tolerance; every supported hidden width */
    MLP_VARIANT_PRIOR_NAIVE = 3, /* training: the paper's baseline, naive 16x16 matmul kernels; comparison only */
    MLP_VARIANT_PRIOR_TILED = 4, /* training: the paper's optimised strategy, tiled + transposed + fused ReLU; comparison only */
    MLP_VARIANT_BF16 = 5,     /* eval and training: as MLP_VARIANT_TF32 with BF16 operands (converted in the kernel, round to
                                 nearest even; tcgen05.mma kind::f16, fp32 accumulate); separately reported, own tolerance */
    MLP_VARIANT_TF32X3 = 6    /* eval only, hidden <= 256: eq. 1 as three TF32 products (X = Xh + Xl, W = Wh + Wl;
                                 Xh Wh + Xl Wh + Xh Wl), fp32-faithful (loss within 1e-5 of the exact value);
                                 separately reported */
};

/*
 * mlp_init -- PAPER.md:98-116.  Records the model descriptor {seed, in, hidden, out}.
 * Supported: in == 32, out == 1, hidden in {32, 64, 128, 256, 512, 1024} (the paper's
 * hidden-width sweep).  Anything else -> MLP_ERR_UNSUPPORTED.  No device work.
 * May be called again to switch model.
 */
int mlp_init(uint64_t seed, int in, int hidden, int out);

/*
 * mlp_init_weights -- fills W1 [in*hidden] and W2 [hidden] (device) with U(+-1/sqrt(fan_in)),
 * fan_in = in for W1 and hidden for W2 (BASELINE.json configs).  Counter-based, so a second
 * implementation can restate it: for flat element index e (W1 row-major, then W2)
 *     z = seed + 0x9E3779B97F4A7C15 * (e + 1)                       (mod 2^64)
 *     z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9
 *     z = (z ^ (z >> 27)) * 0x94D049BB133111EB
 *     z =  z ^ (z >> 31)
 *     u = (z >> 40) * 2^-24 ;   w = (float)((2u - 1) * bound),  bound = 1/sqrt(fan_in) in double.
 * Asynchronous on `stream`.
 */
int mlp_init_weights(float* W1, float* W2, void* stream);

/*
 * mlp_train -- eqs. 1-9 over `epochs` passes of ceil(n/batch) sequential batches
 * (PAPER.md:108-112).  Updates W1/W2 in place; X, Y read-only.  Asynchronous on `stream`
 * (the weights are valid once the stream is synchronised).  epochs == 0 is a no-op.
 * lr == 0 leaves the weights bit-identical.  batch > n is allowed (one short batch per epoch).
 * Equivalent to mlp_train_ex(..., NULL, MLP_VARIANT_FUSED, stream).
 */
int mlp_train(const float* X, const float* Y, int64_t n, int batch, float lr, int epochs,
              float* W1, float* W2, void* stream);

/*
 * mlp_train_ex -- as mlp_train, plus
 *   batch_order: NULL, or device int32 [epochs * nb], nb = ceil(n/batch): step e*nb+k trains on
 *                batch index batch_order[e*nb+k] (BASELINE.json configs 2-5: "batch order a
 *                per-epoch permutation").  Entries must lie in [0, nb).  The device kernels clamp an
 *                out-of-range entry into [0, nb) (no out-of-bounds access) and count it: see
 *                mlp_train_order_errors().  The per-equation variants and the host entry points
 *                validate the table on the host and return MLP_ERR_BAD_ARG before any work.
 *   variant:     MLP_VARIANT_FUSED, MLP_VARIANT_UNFUSED, MLP_VARIANT_PRIOR_NAIVE, MLP_VARIANT_PRIOR_TILED, or
 *                MLP_VARIANT_TF32 (stated tolerance vs the exact path: weights within 5e-5 after one step,
 *                2e-3 after one epoch, loss within 1 %), or MLP_VARIANT_BF16 (1e-4 / 5e-3 / 1 %).
 */
int mlp_train_ex(const float* X, const float* Y, int64_t n, int batch, float lr, int epochs,
                 float* W1, float* W2, const int32_t* batch_order, int variant, void* stream);

/*
 * mlp_train_rows -- mini-batch SGD with SAMPLE-level shuffling (the other reading of "batch order",
 * DESIGN.md reading 5; the paper is silent on shuffling): in epoch e, batch k is
 * rows row_order[e*n + k*batch .. e*n + min(n, (k+1)*batch)) of X/Y.
 *   row_order: DEVICE int32 [epochs*n], each epoch a permutation of 0..n-1 (entries outside [0, n) are
 *              clamped and counted, see mlp_train_order_errors(); duplicates are not detected).
 * Per epoch the rows are gathered into library-owned scratch (one pass at HBM speed) and the fused
 * kernel runs the epoch on the gathered copy: two launches per epoch.  Same arithmetic, same
 * error behaviour and asynchrony as mlp_train; the scratch (n*132 bytes) is freed by mlp_shutdown.
 */
int mlp_train_rows(const float* X, const float* Y, int64_t n, int batch, float lr, int epochs,
                   float* W1, float* W2, const int32_t* row_order, void* stream);

/*
 * mlp_eval_loss -- eq. 4 over the whole dataset:
 *   L = (1/n) sum_r (ReLU(X_r W1) W2 - Y_r)^2.
 * Synchronises `stream` and returns L; NaN on error (then see mlp_last_error()).
 * Deterministic: fp32 inside a row, fp64 from the per-warp partial upwards, fixed tree.
 */
double mlp_eval_loss(const float* X, const float* Y, int64_t n,
                     const float* W1, const float* W2, void* stream);

/* As mlp_eval_loss without the synchronisation: the loss is written to *d_out (device double).
 *   variant: MLP_VARIANT_FUSED = the exact-fp32 kernel of mlp_eval_loss (bound by the FP32 pipes);
 *            MLP_VARIANT_TF32  = eq. 1 on the tensor cores (tcgen05.mma kind::tf32: fp32 operands
 *            truncated to TF32, fp32 accumulate), the HBM-bound variant; stated tolerance: loss within
 *            1 % of the exact value (measured <= 1e-4 relative); n < 2^31 - 128, otherwise MLP_ERR_CUDA.
 *            MLP_VARIANT_BF16  = the same with BF16 operands (rounded to nearest even in the kernel), loss within 1 %;
 *            MLP_VARIANT_TF32X3 = three TF32 products, loss within 1e-5 of the exact value, hidden <= 256
 *            (MLP_ERR_UNSUPPORTED otherwise).  X must be 16-byte aligned.  Deterministic. */
int mlp_eval_loss_async(const float* X, const float* Y, int64_t n, const float* W1,
                        const float* W2, double* d_out, int variant, void* stream);

/*
 * mlp_eval_loss_ws -- mlp_eval_loss_async with a CALLER-owned workspace instead of a pool slot:
 * `workspace` is a device buffer of at least mlp_eval_workspace_bytes() bytes, 8-byte aligned, whose
 * first use must find it zero-filled (the kernel leaves it reusable); launches that may run
 * concurrently need distinct workspaces.  mlp_eval_workspace_bytes() returns 0 without a CUDA device.
 */
size_t mlp_eval_workspace_bytes(void);
int mlp_eval_loss_ws(const float* X, const float* Y, int64_t n, const float* W1, const float* W2,
                     double* d_out, int variant, void* workspace, size_t workspace_bytes, void* stream);

/*
 * mlp_eval_loss_static -- mlp_eval_loss_async for callers that cannot allocate device memory (code
 * under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Same kernels,
 * arguments, variants, results and error behaviour as mlp_eval_loss_async; the per-CTA partial sums
 * and the last-block ticket live in a file-scope __device__ array of the library (8,448 bytes, held
 * by every GPU that loads the library until the process exits) instead of a pool slot.  The call
 * makes no cudaMalloc / cudaFree and creates no events or streams.  The array holds
 * MLP_STATIC_EVAL_MAX_CTAS partial sums; a launch that needs more (one CTA per SM: a device with
 * more SMs than that) returns MLP_ERR_UNSUPPORTED.  ALL calls on a device share the one array:
 * each call clears the ticket on `stream` before its kernel, and two calls whose kernels may
 * overlap on the GPU (different streams without an ordering between them) race -- order them, or
 * use mlp_eval_loss_async / mlp_eval_loss_ws for the concurrent ones.  Calls on one stream are safe.
 */
#define MLP_STATIC_EVAL_MAX_CTAS 1024
int mlp_eval_loss_static(const float* X, const float* Y, int64_t n, const float* W1, const float* W2,
                         double* d_out, int variant, void* stream);

/*
 * Host-buffer entry points (end-to-end path): copy X/Y (and weights / order) from HOST memory
 * to library-owned device buffers, run the same kernels, copy the result back, synchronise.
 * W1_host/W2_host are read and overwritten with the trained weights.  order_host may be NULL; if
 * given, every entry is validated on the host first (MLP_ERR_BAD_ARG, nothing copied or launched).
 *   mlp_train_host      the whole job in one training launch.
 *   mlp_fit_host        BASELINE.json configs[2]: training with "a full-dataset eval-loss pass after
 *                       each epoch" (eq. 4): one training launch and one eval launch (eval_variant) per
 *                       epoch, all asynchronous behind one copy of the dataset; epoch_loss_host [epochs]
 *                       receives the losses (NULL: no evaluation, identical to mlp_train_host).
 *   mlp_eval_loss_host  X/Y are copied in 32 MiB chunks on a second stream and the eval kernel of a
 *                       chunk starts as soon as the chunk has landed (copy and compute overlap; the
 *                       pass is PCIe-bound).  The dataset loss is the row-weighted mean of the per-chunk
 *                       means, formed in chunk order (deterministic); n <= 262,144 rows is one chunk and
 *                       returns exactly what mlp_eval_loss returns.
 */
int mlp_train_host(const float* X_host, const float* Y_host, int64_t n, int batch, float lr,
                   int epochs, float* W1_host, float* W2_host, const int32_t* order_host,
                   int variant);
int mlp_fit_host(const float* X_host, const float* Y_host, int64_t n, int batch, float lr, int epochs,
                 float* W1_host, float* W2_host, const int32_t* order_host, int variant,
                 int eval_variant, double* epoch_loss_host);
double mlp_eval_loss_host(const float* X_host, const float* Y_host, int64_t n,
                          const float* W1_host, const float* W2_host, int variant);

/*
 * Tuning knobs of the fused training kernel.  cluster: number of CTAs (= SMs) the hidden
 * dimension is split over; 0 = automatic.  Valid values are those with hidden/cluster in
 * {16, 32, 64} and cluster in {1, 2, 4, 8, 16}.  Returns MLP_ERR_UNSUPPORTED otherwise.
 */
int mlp_set_cluster(int cluster);
int mlp_get_cluster(void);          /* the cluster size the next mlp_train would use at batch 256 */
int mlp_get_cluster_for(int batch); /* ... at the given batch size (the automatic choice depends on it) */

/*
 * Statistics of the most recently ISSUED fused mlp_train* launch (call after synchronising its
 * stream; concurrent launches each have their own slot, so they do not disturb each other):
 * out[0] = SM clock cycles spent in the kernel (clock64 delta of CTA 0), out[1] = nanoseconds
 * (globaltimer delta), out[2] = SGD steps, out[3] = cluster size.
 */
int mlp_get_train_stats(double out[4]);

/*
 * Number of batch_order / row_order entries of that launch (for mlp_train_rows: of that call) that
 * were outside their valid range and were clamped by the device kernels; 0 for a valid table,
 * -1 on a CUDA error.  Call after synchronising the stream.
 */
int64_t mlp_train_order_errors(void);

/* Number of kernels this library has launched since load (all entry points). */
int64_t mlp_launch_count(void);

const char* mlp_last_error(void);   /* static thread-local string; never NULL */
const char* mlp_version(void);
void mlp_shutdown(void);            /* frees library-owned device scratch; idempotent */

#ifdef __cplusplus
}
#endif
#endif /* PAPER_2606_30497_MLP_H */
