// train_fused.cu -- persistent fused training kernel.
//
// One thread-block cluster of C CTAs (one per SM) runs EVERY SGD step of mlp_train in a single
// launch (PAPER.md:108-112 loop; eqs. 1-9).  The hidden dimension is split over
// the cluster: CTA c owns S = hidden/C hidden units, i.e. W1[:, cS:(c+1)S] and W2[cS:(c+1)S],
// which stay on chip (registers + shared memory) for the whole run.
//
// Mapping inside a CTA (8 warps):
//   * a lane owns TWO hidden units (u0 = lu, u1 = lu + LPS, lu = lane % LPS, LPS = S/2) and keeps
//     their W1 columns (2 x 32 floats) and dW1 accumulators (2 x 32 floats) in registers, as
//     16 + 16 packed fp32x2 pairs over consecutive inputs (i, i+1), so eq. 1 and eq. 8 run on
//     FFMA2 (fma.rn.f32x2): one issue slot per two FMAs;
//   * a warp owns BT/8 rows of the batch tile and walks them SPW = 32/LPS rows at a time; the X
//     row is read from shared memory with broadcast 128-bit loads;
//   * H = ReLU(Z1) for the warp's rows stays in registers between forward and backward.
// Per tile: forward (eqs. 1-3) -> per-row partial Ypred reduced across the LPS lanes with a
// transposing shuffle tree -> pushed to every CTA of the cluster with st.async (DSMEM store that
// completes transaction bytes on the destination's mbarrier: one hop, no flag) -> every CTA sums
// the C partials in rank order -> dZ2 (eq. 5) -> dW2, dZ1, dW1 (eqs. 6-8) accumulated in
// registers.  The tile is processed as NSPLIT row groups so that the exchange of one group is in
// flight while the other group computes.  At the end of the batch the 8 warps' partial gradients
// are summed through shared memory in a fixed order (deterministic), eq. 9 is applied to the
// shared-memory master copy and the warps re-load their columns.
// X tiles arrive by cp.async.bulk (TMA engine) into a 2-deep ring, one tile ahead; batches with
// more than BT rows are processed as several tiles with the gradients kept in registers.
#include "common.cuh"
#include "internal.h"

namespace mlp {
namespace {

constexpr int kWarps = 8;
constexpr int kThreads = kWarps * 32;

struct TrainParams {
    const float* X;
    const float* Y;
    long long n;
    int B;
    float lr;
    long long total_steps;
    long long nb;
    float* W1;
    float* W2;
    const int* order;
    int H;
    unsigned long long* stats;
};

// Sum NV per-lane values across the L lanes of a sample group.  On return v[0] of the lane with
// (lu & (NV-1)) == k holds the total of original entry k (transposing butterfly: each step halves
// the number of live values, so the whole reduction costs NV-1 + log2(L/NV) shuffles).
template <int NV, int L, int O = 1>
struct GroupReduce {
    static __device__ __forceinline__ void run(float* v, int lu) {
        if constexpr (NV > 1) {
            const bool up = (lu & O) != 0;
#pragma unroll
            for (int k = 0; k < NV / 2; ++k) {
                const float keep = up ? v[2 * k + 1] : v[2 * k];
                const float send = up ? v[2 * k] : v[2 * k + 1];
                v[k] = keep + __shfl_xor_sync(0xffffffffu, send, O);
            }
            GroupReduce<NV / 2, L, O * 2>::run(v, lu);
        } else if constexpr (O < L) {
            v[0] += __shfl_xor_sync(0xffffffffu, v[0], O);
            GroupReduce<1, L, O * 2>::run(v, lu);
        }
    }
};

__device__ __forceinline__ f32x2 shfl_xor2(f32x2 v, int o) {
    return __shfl_xor_sync(0xffffffffu, v, o);
}

template <int S, int BT, int NSPLIT>
__global__ void __launch_bounds__(kThreads, 1) k_train_fused(const TrainParams p) {
    constexpr int LPS = S / 2;            // lanes per sample row
    constexpr int SPW = 32 / LPS;         // sample rows per warp instruction
    constexpr int RPW = BT / kWarps;      // rows per warp per tile
    constexpr int ITER = RPW / SPW;       // row groups per warp per tile
    constexpr int ITS = ITER / NSPLIT;    // row groups per exchange sub-tile
    static_assert(LPS >= 8 && LPS <= 32 && RPW % SPW == 0 && ITER % NSPLIT == 0 && ITS >= 1, "cfg");
    static_assert(ITS <= LPS, "transposing reduction needs ITS <= LPS");

    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int lu = lane % LPS, s = lane / LPS;
    const uint32_t crank = cluster_ctarank(), C = cluster_nctarank();
    const int H = p.H;

    float* Xs = reinterpret_cast<float*>(smem_raw);          // [2][BT*32]
    float* ypp = Xs + 2 * BT * kIn;                           // [2][C][BT]
    float* part = ypp + 2 * C * BT;                           // [kWarps][S*32]  layout [q][u][4]
    float* part2 = part + kWarps * S * kIn;                   // [kWarps][S]
    float* W1s = part2 + kWarps * S;                          // [S*32]          layout [q][u][4]
    float* W2s = W1s + S * kIn;                               // [S]
    uint64_t* bars = reinterpret_cast<uint64_t*>(W2s + S);    // full[2], empty[2], yp[2][NSPLIT]
    const uint32_t bar_full = smem_u32(bars), bar_empty = smem_u32(bars + 2),
                   bar_yp = smem_u32(bars + 4);

    unsigned long long clk0 = 0, ns0 = 0;
    if (crank == 0 && tid == 0) { clk0 = clock64(); ns0 = globaltimer_ns(); }

    // ---- one-time setup: zero the X ring, load this CTA's weight slice, init barriers ----------
    for (int f = tid; f < 2 * BT * kIn; f += kThreads) Xs[f] = 0.f;
    for (int f = tid; f < S * kIn; f += kThreads) {
        const int q = f / (S * 4), rem = f % (S * 4), u = rem >> 2, i = q * 4 + (rem & 3);
        W1s[f] = p.W1[(size_t)i * H + crank * S + u];
    }
    if (tid < S) W2s[tid] = p.W2[crank * S + tid];
    if (tid == 0) {
        for (int b = 0; b < 2; ++b) {
            mbar_init(bar_full + 8 * b, 1);
            mbar_init(bar_empty + 8 * b, kWarps);
            for (int q = 0; q < NSPLIT; ++q) mbar_init(bar_yp + 8 * (b * NSPLIT + q), 1);
        }
        fence_mbar_init();
    }
    // generic-proxy zero fill of Xs must be ordered before the async-proxy bulk copies
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();
    cluster_sync_all();        // every CTA's barriers exist before anyone pushes to them

    // ---- per-lane weight registers ---------------------------------------------------------------
    f32x2 w0[16], w1[16];      // W1 columns of u0, u1 as (i, i+1) pairs
    float w2r0, w2r1;
    auto reload_weights = [&]() {
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const ulonglong2 a = *reinterpret_cast<const ulonglong2*>(W1s + (q * S + lu) * 4);
            const ulonglong2 b = *reinterpret_cast<const ulonglong2*>(W1s + (q * S + lu + LPS) * 4);
            w0[2 * q] = a.x; w0[2 * q + 1] = a.y;
            w1[2 * q] = b.x; w1[2 * q + 1] = b.y;
        }
        w2r0 = W2s[lu];
        w2r1 = W2s[lu + LPS];
    };
    reload_weights();

    const long long total = p.total_steps;
    auto batch_index = [&](long long step) -> int {
        return p.order ? __ldg(p.order + step) : (int)(step % p.nb);
    };
    int t_cur = batch_index(0);
    int t_next = total > 1 ? batch_index(1) : 0;

    // producer state: issue tile 0
    if (warp == 0 && lane == 0) {
        const long long r0 = (long long)t_cur * p.B;
        const int m = (int)min((long long)p.B, p.n - r0);
        const int rows = min(BT, m);
        mbar_arrive_expect_tx(bar_full, rows * 128);
        bulk_g2s(smem_u32(Xs), p.X + r0 * kIn, rows * 128, bar_full);
    }

    unsigned gt = 0;   // global tile counter
    for (long long step = 0; step < total; ++step) {
        const int t_nn = (step + 2 < total) ? batch_index(step + 2) : 0;
        const long long r0 = (long long)t_cur * p.B;
        const int m = (int)min((long long)p.B, p.n - r0);
        const int ntiles = (m + BT - 1) / BT;
        const float scale = 2.0f / (float)m;                  // eq. 5

        f32x2 acc0[16], acc1[16];                             // dW1 partials of u0, u1 (eq. 8)
#pragma unroll
        for (int k = 0; k < 16; ++k) { acc0[k] = 0ull; acc1[k] = 0ull; }
        float g20 = 0.f, g21 = 0.f;                           // dW2 partials (eq. 6)

        for (int j = 0; j < ntiles; ++j, ++gt) {
            const unsigned buf = gt & 1u, ph = (gt >> 1) & 1u;
            const int vt = min(BT, m - j * BT);               // valid rows in this tile
            const float* Xt = Xs + buf * (BT * kIn);
            const float* ypt = ypp + buf * (C * BT);

            if (warp == 0 && lane == 0) {
                // arm this tile's exchange barriers
#pragma unroll
                for (int q = 0; q < NSPLIT; ++q)
                    mbar_arrive_expect_tx(bar_yp + 8 * (buf * NSPLIT + q), C * (BT / NSPLIT) * 4);
                // prefetch the next tile into the other buffer
                long long nr0; int nrows; bool have = true;
                if (j + 1 < ntiles) { nr0 = r0 + (long long)(j + 1) * BT; nrows = min(BT, m - (j + 1) * BT); }
                else if (step + 1 < total) {
                    nr0 = (long long)t_next * p.B;
                    nrows = (int)min((long long)min(BT, p.B), p.n - nr0);
                } else { have = false; nr0 = 0; nrows = 0; }
                if (have) {
                    const unsigned g1 = gt + 1, nbuf = g1 & 1u;
                    if (g1 >= 2) mbar_wait(bar_empty + 8 * nbuf, ((g1 >> 1) - 1) & 1u);
                    mbar_arrive_expect_tx(bar_full + 8 * nbuf, nrows * 128);
                    bulk_g2s(smem_u32(Xs + nbuf * (BT * kIn)), p.X + nr0 * kIn, nrows * 128,
                             bar_full + 8 * nbuf);
                }
            }
            __syncwarp();

            // targets of the rows whose dZ2 this lane will compute (latency hidden by the forward)
            float yv[NSPLIT];
#pragma unroll
            for (int q = 0; q < NSPLIT; ++q) {
                const int row = warp * RPW + (q * ITS + (lu & (ITS - 1))) * SPW + s;
                yv[q] = row < vt ? __ldg(p.Y + r0 + (long long)j * BT + row) : 0.f;
            }

            mbar_wait(bar_full + 8 * buf, ph);

            // ---------------- forward: eqs. 1-3 ----------------
            float hreg[ITER][2];
#pragma unroll
            for (int q = 0; q < NSPLIT; ++q) {
                float pv[ITS];
#pragma unroll
                for (int k = 0; k < ITS; ++k) {
                    const int it = q * ITS + k;
                    const int row = warp * RPW + it * SPW + s;
                    const ulonglong2* xrow = reinterpret_cast<const ulonglong2*>(Xt + row * kIn);
                    f32x2 a0 = 0ull, a1 = 0ull;
#pragma unroll
                    for (int x = 0; x < 8; ++x) {
                        const ulonglong2 xv = xrow[x];
                        ffma2(a0, xv.x, w0[2 * x]); ffma2(a1, xv.x, w1[2 * x]);
                        ffma2(a0, xv.y, w0[2 * x + 1]); ffma2(a1, xv.y, w1[2 * x + 1]);
                    }
                    const bool valid = row < vt;
                    const float h0 = valid ? fmaxf(hsum2(a0), 0.f) : 0.f;     // eq. 2
                    const float h1 = valid ? fmaxf(hsum2(a1), 0.f) : 0.f;
                    hreg[it][0] = h0; hreg[it][1] = h1;
                    pv[k] = fmaf(h1, w2r1, h0 * w2r0);                        // eq. 3 (partial)
                }
                GroupReduce<ITS, LPS>::run(pv, lu);
                if (lu < ITS) {
                    const int row = warp * RPW + (q * ITS + lu) * SPW + s;
                    const uint32_t dst = smem_u32(ypp + buf * (C * BT) + crank * BT + row);
                    const uint32_t bar = bar_yp + 8 * (buf * NSPLIT + q);
                    for (uint32_t dd = 0; dd < C; ++dd) {
                        const uint32_t d = (crank + dd) % C;
                        st_async_f32(mapa(dst, d), pv[0], mapa(bar, d));
                    }
                }
            }

            // ---------------- backward: eqs. 5-8 ----------------
#pragma unroll
            for (int q = 0; q < NSPLIT; ++q) {
                mbar_wait_cluster(bar_yp + 8 * (buf * NSPLIT + q), ph);
                float dzv;
                {
                    const int row = warp * RPW + (q * ITS + (lu & (ITS - 1))) * SPW + s;
                    float yp = 0.f;
                    for (uint32_t c = 0; c < C; ++c) yp += ypt[c * BT + row];  // fixed rank order
                    dzv = row < vt ? scale * (yp - yv[q]) : 0.f;              // eq. 5
                }
#pragma unroll
                for (int k = 0; k < ITS; ++k) {
                    const int it = q * ITS + k;
                    const int row = warp * RPW + it * SPW + s;
                    const float d = __shfl_sync(0xffffffffu, dzv, (lane & ~(LPS - 1)) | k);
                    const float h0 = hreg[it][0], h1 = hreg[it][1];
                    g20 = fmaf(h0, d, g20);                                    // eq. 6
                    g21 = fmaf(h1, d, g21);
                    const float e0 = h0 > 0.f ? d * w2r0 : 0.f;                // eq. 7 (old W2)
                    const float e1 = h1 > 0.f ? d * w2r1 : 0.f;
                    const f32x2 dd0 = pack2(e0, e0), dd1 = pack2(e1, e1);
                    const ulonglong2* xrow = reinterpret_cast<const ulonglong2*>(Xt + row * kIn);
#pragma unroll
                    for (int x = 0; x < 8; ++x) {                              // eq. 8
                        const ulonglong2 xv = xrow[x];
                        ffma2(acc0[2 * x], xv.x, dd0); ffma2(acc1[2 * x], xv.x, dd1);
                        ffma2(acc0[2 * x + 1], xv.y, dd0); ffma2(acc1[2 * x + 1], xv.y, dd1);
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_empty + 8 * buf);   // this warp is done with the X tile
        }

        // ---------------- end of batch: reduce partial gradients, eq. 9 ----------------
        if constexpr (SPW > 1) {
            const f32x2 one = pack2(1.f, 1.f);
#pragma unroll
            for (int o = LPS; o < 32; o <<= 1) {
#pragma unroll
                for (int k = 0; k < 16; ++k) {
                    ffma2(acc0[k], shfl_xor2(acc0[k], o), one);
                    ffma2(acc1[k], shfl_xor2(acc1[k], o), one);
                }
                g20 += __shfl_xor_sync(0xffffffffu, g20, o);
                g21 += __shfl_xor_sync(0xffffffffu, g21, o);
            }
        }
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            // after the reduction every sub-sample group holds the sums: spread the stores
            if (s == (q * SPW) / 16)
                *reinterpret_cast<ulonglong2*>(part + ((warp * 8 + q) * S + lu) * 4) =
                    make_ulonglong2(acc0[2 * q], acc0[2 * q + 1]);
            if (s == ((8 + q) * SPW) / 16)
                *reinterpret_cast<ulonglong2*>(part + ((warp * 8 + q) * S + lu + LPS) * 4) =
                    make_ulonglong2(acc1[2 * q], acc1[2 * q + 1]);
        }
        if (s == 0) { part2[warp * S + lu] = g20; part2[warp * S + lu + LPS] = g21; }
        __syncthreads();
        for (int f = tid; f < S * 8; f += kThreads) {
            float4 sum = reinterpret_cast<const float4*>(part)[f];
#pragma unroll
            for (int w = 1; w < kWarps; ++w) {
                const float4 v = reinterpret_cast<const float4*>(part)[w * S * 8 + f];
                sum.x += v.x; sum.y += v.y; sum.z += v.z; sum.w += v.w;
            }
            float4 wv = reinterpret_cast<float4*>(W1s)[f];
            wv.x -= p.lr * sum.x; wv.y -= p.lr * sum.y; wv.z -= p.lr * sum.z; wv.w -= p.lr * sum.w;
            reinterpret_cast<float4*>(W1s)[f] = wv;                            // eq. 9
        }
        if (tid < S) {
            float sum = part2[tid];
#pragma unroll
            for (int w = 1; w < kWarps; ++w) sum += part2[w * S + tid];
            W2s[tid] -= p.lr * sum;                                            // eq. 9
        }
        __syncthreads();
        reload_weights();
        t_cur = t_next;
        t_next = t_nn;
    }

    // ---- write the trained slice back to the caller's buffers ------------------------------------
    for (int f = tid; f < S * kIn; f += kThreads) {
        const int q = f / (S * 4), rem = f % (S * 4), u = rem >> 2, i = q * 4 + (rem & 3);
        p.W1[(size_t)i * H + crank * S + u] = W1s[f];
    }
    if (tid < S) p.W2[crank * S + tid] = W2s[tid];
    if (crank == 0 && tid == 0 && p.stats) {
        p.stats[0] = clock64() - clk0;
        p.stats[1] = globaltimer_ns() - ns0;
        p.stats[2] = (unsigned long long)total;
        p.stats[3] = C;
    }
    cluster_sync_all();        // no CTA exits while peers may still push into its shared memory
}

template <int S, int BT, int NSPLIT>
cudaError_t launch_cfg(const TrainParams& p, int cluster, cudaStream_t stream) {
    auto kern = k_train_fused<S, BT, NSPLIT>;
    const size_t smem = sizeof(float) * (2 * BT * kIn + 2 * cluster * BT + kWarps * S * kIn +
                                         kWarps * S + S * kIn + S) + 8 * (4 + 2 * NSPLIT);
    cudaError_t err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err != cudaSuccess) return err;
    if (cluster > 8) {
        err = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (err != cudaSuccess) return err;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(cluster);
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = cluster;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, p);
}

template <int S>
cudaError_t launch_s(const TrainParams& p, int cluster, cudaStream_t stream) {
    const int B = p.B;
    if (B > 128) return launch_cfg<S, 256, 2>(p, cluster, stream);
    if (B > 64) return launch_cfg<S, 128, 2>(p, cluster, stream);
    if (B > 32) return launch_cfg<S, 64, (64 / kWarps) / (64 / S) >= 4 ? 2 : 1>(p, cluster, stream);
    return launch_cfg<S, 32, 1>(p, cluster, stream);
}

}  // namespace

bool fused_supported(int hidden, int cluster) {
    if (cluster != 1 && cluster != 2 && cluster != 4 && cluster != 8 && cluster != 16) return false;
    if (hidden % cluster) return false;
    const int S = hidden / cluster;
    return S == 16 || S == 32 || S == 64;
}

int fused_default_cluster(int hidden) {
    switch (hidden) {
        case 32: return 1;
        case 64: return 2;
        case 128: return 4;
        case 256: return 8;
        case 512: return 16;
        case 1024: return 16;
        default: return 0;
    }
}

cudaError_t launch_train_fused(const float* X, const float* Y, int64_t n, int batch, float lr,
                               int epochs, float* W1, float* W2, const int32_t* order,
                               int hidden, int cluster, unsigned long long* stats,
                               cudaStream_t stream, int64_t* launches) {
    TrainParams p;
    p.X = X; p.Y = Y; p.n = n; p.B = batch; p.lr = lr;
    p.nb = (n + batch - 1) / batch;
    p.total_steps = (long long)epochs * p.nb;
    p.W1 = W1; p.W2 = W2; p.order = order; p.H = hidden; p.stats = stats;
    if (p.total_steps == 0) return cudaSuccess;
    cudaError_t err;
    switch (hidden / cluster) {
        case 16: err = launch_s<16>(p, cluster, stream); break;
        case 32: err = launch_s<32>(p, cluster, stream); break;
        case 64: err = launch_s<64>(p, cluster, stream); break;
        default: return cudaErrorInvalidValue;
    }
    if (err == cudaSuccess) ++*launches;
    return err;
}

}  // namespace mlp
