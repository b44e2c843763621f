// eval_fp32.cu -- grid-wide streaming forward + MSE (SURVEY.md 8(a) row a-E), exact fp32.
//
// L = (1/n) sum_r (ReLU(X_r W1) W2 - Y_r)^2     (eqs. 1-4)
//
// Persistent grid (a multiple of the SM count).  Each CTA keeps ALL of W1/W2 in registers
// (a lane owns four hidden units: 4 x 32 weights as packed fp32x2 pairs, as in train_fused.cu)
// and streams 128-row tiles of X (16 KB, one cp.async.bulk each) through a 4-stage
// shared-memory ring.  LPS = hidden/2 lanes cooperate on one row; the X row is read with
// broadcast 128-bit loads and eq. 1 runs on FFMA2.  Per-row partial Ypred values are reduced
// across lanes with a transposing shuffle tree, across the warps of a row group through shared
// memory.  Squared errors accumulate in fp64 per lane; a fixed-order block reduction and a
// fixed-order last-block pass make the result deterministic (no floating-point atomics).
// With exact fp32 FMAs this kernel is bound by the FP32 pipes, not by HBM (128 FLOP/B).
#include "common.cuh"
#include "internal.h"

namespace mlp {
namespace {

constexpr int kTileRows = 128;
constexpr int kStages = 4;

template <int H>
struct EvalCfg {
    static constexpr int LPS = H / 4;                               // lanes per row (four hidden units per lane)
    static constexpr int NT = LPS > 256 ? LPS : 256;                // threads per CTA
    static constexpr int G = NT / LPS;                              // row groups per CTA
    static constexpr int WPG = LPS >= 32 ? LPS / 32 : 1;            // warps per row group
    static constexpr int LW = LPS >= 32 ? 32 : LPS;                 // lanes of one warp on a row
    static constexpr int RPG = kTileRows / G;                       // rows per group per tile
    static constexpr int CH = RPG < 32 ? RPG : 32;                  // rows per reduction chunk
    static constexpr int NCH = RPG / CH;
    static constexpr size_t smem = (size_t)kStages * kTileRows * kIn * 4 +
                                   (size_t)2 * G * WPG * CH * 4 + 8 * 2 * kStages + NT / 32 * 8;
};

template <int H>
__global__ void __launch_bounds__(EvalCfg<H>::NT, 1)
k_eval_fp32(const float* __restrict__ X, const float* __restrict__ Y, long long n,
            const float* __restrict__ W1, const float* __restrict__ W2,
            double* __restrict__ partials, unsigned int* __restrict__ ticket,
            double* __restrict__ out) {
    using Cf = EvalCfg<H>;
    constexpr int LPS = Cf::LPS, NT = Cf::NT, WPG = Cf::WPG, LW = Cf::LW, RPG = Cf::RPG,
                  CH = Cf::CH, NCH = Cf::NCH, G = Cf::G, NWARP = NT / 32;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* Xs = reinterpret_cast<float*>(smem_raw);                       // [kStages][128*32]
    float* red = Xs + kStages * kTileRows * kIn;                          // [2][G][WPG][CH]
    uint64_t* bars = reinterpret_cast<uint64_t*>(red + 2 * G * WPG * CH); // full[], empty[]
    double* wsum = reinterpret_cast<double*>(bars + 2 * kStages);         // [NWARP]
    const uint32_t bar_full = smem_u32(bars), bar_empty = smem_u32(bars + kStages);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    __shared__ int last_flag_s;
    int* last_flag = &last_flag_s;
    const int g = tid / LPS;                 // row group of this thread
    const int gl = tid % LPS;                // lane index inside the group -> hidden units
    const int lu = lane % LW;                // lane index inside the warp's part of the group
    const int wig = (tid % LPS) / 32;        // warp index inside the group

    if (tid == 0) {
        for (int st = 0; st < kStages; ++st) {
            mbar_init(bar_full + 8 * st, 1);
            mbar_init(bar_empty + 8 * st, NWARP);
        }
        fence_mbar_init();
    }
    __syncthreads();

    const long long ntiles = (n + kTileRows - 1) / kTileRows;
    const long long my_tiles = blockIdx.x < ntiles ? (ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    auto issue = [&](long long i) {        // thread 0: load this CTA's i-th tile into stage i % kStages
        const long long tile = blockIdx.x + i * (long long)gridDim.x;
        const long long row0 = tile * kTileRows;
        const int rows = (int)min((long long)kTileRows, n - row0);
        const int st = (int)(i % kStages);
        mbar_arrive_expect_tx(bar_full + 8 * st, rows * 128);
        bulk_g2s(smem_u32(Xs + st * kTileRows * kIn), X + row0 * kIn, rows * 128, bar_full + 8 * st);
    };
    if (tid == 0)
        for (long long i = 0; i < kStages && i < my_tiles; ++i) issue(i);

    // weights: units gl + j*LPS, j < 4: one 128-bit load of X then feeds 8 FFMA2 (4 with two units per
    // lane, where the shared-memory pipe and the FMA pipe saturated together)
    f32x2 w[4][16];
    float w2r[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
#pragma unroll
        for (int k = 0; k < 16; ++k)
            w[j][k] = pack2(W1[(size_t)(2 * k) * H + gl + j * LPS], W1[(size_t)(2 * k + 1) * H + gl + j * LPS]);
        w2r[j] = W2[gl + j * LPS];
    }

    double sse = 0.0;
    unsigned chunk_par = 0;
    for (long long i = 0; i < my_tiles; ++i) {
        const int st = (int)(i % kStages);
        const unsigned ph = (unsigned)((i / kStages) & 1);
        // refill, two tiles behind, the stage every warp has released
        if (tid == 0 && i >= 2 && i - 2 + kStages < my_tiles) {
            const long long j = i - 2;
            mbar_wait(bar_empty + 8 * (int)(j % kStages), (unsigned)((j / kStages) & 1));
            issue(j + kStages);
        }
        __syncwarp();
        const long long tile = blockIdx.x + i * (long long)gridDim.x;
        const long long row0 = tile * kTileRows;
        const int vt = (int)min((long long)kTileRows, n - row0);
        mbar_wait(bar_full + 8 * st, ph);
        const float* Xt = Xs + st * kTileRows * kIn;
#pragma unroll 1
        for (int ch = 0; ch < NCH; ++ch) {
            const int rbase = g * RPG + ch * CH;
            // target of the row this lane finalises (issued early; used after the reduction)
            const int myrow = rbase + (lu & (CH - 1));
            const float yv = myrow < vt ? __ldg(Y + row0 + myrow) : 0.f;
            float pv[CH];
#pragma unroll
            for (int k = 0; k < CH; ++k) {
                const ulonglong2* xrow = reinterpret_cast<const ulonglong2*>(Xt + (rbase + k) * kIn);
                f32x2 a[4];
#pragma unroll
                for (int x = 0; x < 8; ++x) {
                    const ulonglong2 xv = xrow[x];
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        if (x == 0) a[j] = fmul2(xv.x, w[j][0]);                        // eq. 1
                        else ffma2(a[j], xv.x, w[j][2 * x]);
                        ffma2(a[j], xv.y, w[j][2 * x + 1]);
                    }
                }
                float h[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) h[j] = fmaxf(hsum2(a[j]), 0.f);             // eq. 2
                pv[k] = fmaf(h[1], w2r[1], h[0] * w2r[0]) + fmaf(h[3], w2r[3], h[2] * w2r[2]);   // eq. 3
            }
            GroupReduce<CH, LW>::run(pv, lu);
            float yp = pv[0];
            if constexpr (WPG > 1) {
                float* rbuf = red + ((chunk_par * G + g) * WPG) * CH;
                if (lu < CH) rbuf[wig * CH + lu] = yp;
                asm volatile("bar.sync %0, %1;" ::"r"(1 + g), "r"(WPG * 32) : "memory");
                if (wig == 0) {
                    yp = rbuf[lu & (CH - 1)];
#pragma unroll
                    for (int w = 1; w < WPG; ++w) yp += rbuf[w * CH + (lu & (CH - 1))];
                }
                chunk_par ^= 1u;
            }
            if (wig == 0 && lu < CH && myrow < vt) {
                const float e = yp - yv;
                sse += (double)(e * e);                                                // eq. 4
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8 * st);
    }

    // fixed-order reduction: lanes -> warp -> CTA -> grid (last block)
    for (int o = 16; o > 0; o >>= 1) sse += __shfl_down_sync(0xffffffffu, sse, o);
    if (lane == 0) wsum[warp] = sse;
    __syncthreads();
    if (tid == 0) {
        double tot = 0.0;
        for (int w = 0; w < NWARP; ++w) tot += wsum[w];
        partials[blockIdx.x] = tot;
        __threadfence();
        const unsigned prev = atomicAdd(ticket, 1u);
        *last_flag = prev == gridDim.x - 1 ? 1 : 0;
    }
    __syncthreads();
    // last block: fixed-order sum of the per-block partials; the loads of one warp are in flight together
    // (a one-thread loop would pay one L2 round trip per block)
    if (*last_flag && warp == 0) {
        __threadfence();
        double acc = 0.0;
        for (unsigned b = lane; b < gridDim.x; b += 32) acc += ((volatile double*)partials)[b];
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
        if (lane == 0) {
            *out = acc / (double)n;
            *ticket = 0u;
        }
    }
}

template <int H>
cudaError_t launch_h(const float* X, const float* Y, long long n, const float* W1, const float* W2,
                     double* partials, unsigned int* ticket, int grid, double* d_out, cudaStream_t stream) {
    auto kern = k_eval_fp32<H>;
    cudaError_t err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           (int)EvalCfg<H>::smem);
    if (err != cudaSuccess) return err;
    kern<<<grid, EvalCfg<H>::NT, EvalCfg<H>::smem, stream>>>(X, Y, n, W1, W2, partials, ticket, d_out);
    return cudaGetLastError();
}

}  // namespace

int eval_fp32_grid(int hidden, int num_sms) {
    (void)hidden;
    return num_sms;            // one persistent CTA per SM (registers: 1 CTA/SM)
}

cudaError_t launch_eval_fp32(const float* X, const float* Y, int64_t n, const float* W1,
                             const float* W2, int hidden, double* partials, unsigned int* ticket, int grid,
                             double* d_out, cudaStream_t stream, int64_t* launches) {
    cudaError_t err;
    switch (hidden) {
        case 32: err = launch_h<32>(X, Y, n, W1, W2, partials, ticket, grid, d_out, stream); break;
        case 64: err = launch_h<64>(X, Y, n, W1, W2, partials, ticket, grid, d_out, stream); break;
        case 128: err = launch_h<128>(X, Y, n, W1, W2, partials, ticket, grid, d_out, stream); break;
        case 256: err = launch_h<256>(X, Y, n, W1, W2, partials, ticket, grid, d_out, stream); break;
        case 512: err = launch_h<512>(X, Y, n, W1, W2, partials, ticket, grid, d_out, stream); break;
        case 1024: err = launch_h<1024>(X, Y, n, W1, W2, partials, ticket, grid, d_out, stream); break;
        default: return cudaErrorInvalidValue;
    }
    if (err == cudaSuccess) ++*launches;
    return err;
}

}  // namespace mlp
