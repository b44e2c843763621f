// train_tf32.cu -- tensor-core variant of the fused training kernel (SURVEY.md 8(a) row a-T,
// 8(f) NEXT-2; BASELINE.json: "allowed only as a separately reported variant with its own stated
// tolerance").  Same method, same loop, same cluster layout and Ypred exchange as train_fused.cu
// (eqs. 1-9; one launch for every batch of every epoch), but both large products
// run on the tensor cores (tcgen05.mma kind::tf32: fp32 operands truncated to TF32, fp32
// accumulate in TMEM):
//   eq. 1  Z1 = X W1        per 256-row tile two chains M=128 (rows), N=32 (units of this CTA), K=32;
//   eq. 8  dW1^T = dZ1^T X  one chain M=64 (32 units + padding), N=32 (inputs), K=256 rows, in TMEM
//                           across the tiles of a batch.
// Everything else stays fp32 on the CUDA cores.  32 hidden units per CTA: hidden 32..256 on a
// cluster of hidden/32 CTAs (the exchange buffers of a 16-CTA cluster no longer fit beside the
// operands of eq. 8 in shared memory; hidden 1024 would need 32 CTAs per cluster).
//
// Per tile and CTA (8 warps, a thread owns ONE row of the tile):
//   TMA (cp.async.bulk.tensor, 128-byte swizzle) brings the X tile [256 x 32] one tile ahead; warp 0
//   issues eq. 1 (A = X tile as delivered, B = W1^T slice in operand layout); while it runs every thread
//   transposes its X row into the K-major B operand of eq. 8; then it reads its 32 pre-activations
//   from TMEM, applies eq. 2, stores H, forms its partial of eq. 3 and pushes it to the 8 CTAs
//   (st.async + mbarrier); after the exchange it computes dZ2 (eq. 5) and writes its row of
//   dZ1 = dZ2 ReLU'(Z1) W2 (eq. 7) into the K-major A operand of eq. 8; warp 0 issues eq. 8 while all
//   warps do eq. 6 (dW2) on the CUDA cores.  At the end of the batch the 32 threads that own the TMEM
//   rows of dW1^T (one per hidden unit) apply eq. 9 to the fp32 master row they keep in registers and
//   rewrite their row of the eq. 1 operand.  No W1 register reload, no CUDA-core backward loop.
// All operands are K-major with the 128-byte swizzle (the conventions of eval_tf32.cu).
#include <cuda.h>

#include "tc_common.cuh"

namespace mlp {
namespace {

constexpr int kS = 32;            // hidden units per CTA
// cluster size C = hidden / 32 is a template parameter (1, 2, 4 or 8)
constexpr int kBT = 256;          // rows per tile
constexpr int kWarps = 8;
constexpr int kThreads = kWarps * 32;
constexpr int kRing = 2;          // X ring stages (the operands of eq. 8 take the rest of shared memory)
constexpr uint32_t kXBytes = kBT * kIn * 4;

struct TcParams {
    const float* Y;
    long long n;
    int B;
    float lr;
    long long total_steps;
    int nbi, m_last;
    float scale_full, scale_last;
    float* W1;
    float* W2;
    const int* order;
    int H;
    unsigned long long* stats;   // [4] = batch_order entries outside [0, nb) (clamped and counted)
};

template <int C>
__global__ void __launch_bounds__(kThreads, 1)
k_train_tf32(const __grid_constant__ CUtensorMap tmapX, const TcParams p) {
    constexpr int S = kS, BT = kBT;
    constexpr int NA = BT / 32;                                           // 32-row K atoms of the backward product
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char* Xs = smem;                                             // [kRing][32 KB] X tiles, swizzled rows (A of eq. 1)
    unsigned char* Wop = Xs + kRing * kXBytes;                            // [S][128 B] W1^T slice (B of eq. 1), K-major swizzled
    unsigned char* At = Wop + S * 128;                                    // [NA][64][128 B] dZ1^T (A of eq. 8), rows 32-63 padding
    unsigned char* Xt = At + NA * 64 * 128;                               // [NA][32][128 B] X^T (B of eq. 8)
    unsigned char* Hs = Xt + NA * 32 * 128;                               // [BT][128 B] H = ReLU(Z1), swizzled rows (eq. 6)
    float* ypp = reinterpret_cast<float*>(Hs + BT * 128);                 // [2][C][BT]
    float* part2 = ypp + 2 * C * BT;                                      // [kWarps][S] dW2 partials
    float* W2s = part2 + kWarps * S;                                      // [S]
    float* Ds = W2s + S;                                                  // [BT] dZ2 of the tile
    uint64_t* bars = reinterpret_cast<uint64_t*>(Ds + BT);                // full[3], empty[3], yp[2], mma, mma2
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * kRing + 4);
    const uint32_t bar_full = smem_u32(bars), bar_empty = smem_u32(bars + kRing),
                   bar_yp = smem_u32(bars + 2 * kRing), bar_mma = smem_u32(bars + 2 * kRing + 2),
                   bar_mma2 = smem_u32(bars + 2 * kRing + 3);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t crank = cluster_ctarank();
    const int H = p.H;
    // forward ownership: thread <-> tile row (TMEM lane rule: warp w reads lanes 32*(w%4)..)
    const int frow = (warp >> 2) * 128 + (warp & 3) * 32 + lane;
    // weight ownership: the M=64 accumulator of eq. 8 keeps unit u in TMEM lane (u/16)*32 + u%16, i.e. lanes
    // 0-15 of warps 0 and 1: those 32 threads hold the fp32 master row W1[:, u] in registers for the whole run
    const bool wowner = warp < 2 && lane < 16;
    const int wu = warp * 16 + lane;                                      // owned hidden unit (if wowner)
    float wrow[kIn];
#pragma unroll
    for (int i = 0; i < kIn; ++i) wrow[i] = wowner ? p.W1[(size_t)i * H + crank * S + wu] : 0.f;
    auto store_wop = [&]() {                                              // B[n = u][k = i], eq. 1 operand
#pragma unroll
        for (int c = 0; c < 8; ++c)
            *reinterpret_cast<float4*>(Wop + swz(wu, c)) = make_float4(wrow[4 * c], wrow[4 * c + 1], wrow[4 * c + 2], wrow[4 * c + 3]);
    };

    // ---- one-time setup ---------------------------------------------------------------------------
    if (wowner) store_wop();
    for (int f = tid; f < NA * 64 * 32; f += kThreads) reinterpret_cast<float*>(At)[f] = 0.f;   // padding rows stay 0
    if (tid < S) W2s[tid] = p.W2[crank * S + tid];
    if (tid == 0) {
        for (int b = 0; b < kRing; ++b) { mbar_init(bar_full + 8 * b, 1); mbar_init(bar_empty + 8 * b, kWarps); }
        mbar_init(bar_yp, 1); mbar_init(bar_yp + 8, 1); mbar_init(bar_mma, 1); mbar_init(bar_mma2, 1);
        fence_mbar_init();
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 128;" ::"r"(smem_u32(tmem_slot)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");          // generic writes -> MMA (async proxy)
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    if (smem_u32(smem) & 1023u) __trap();
    cluster_sync_all();        // every CTA's barriers exist before anyone pushes to them

    const long long total = p.total_steps;
    int seq = 0;
    unsigned long long bad_order = 0;     // batch_order entries outside [0, nb): clamped, counted, reported
    auto batch_index = [&](long long step, int sq) -> int {
        if (!p.order) return sq;
        const int t = __ldg(p.order + step);
        if ((unsigned)t < (unsigned)p.nbi) return t;
        ++bad_order;
        return t < 0 ? 0 : p.nbi - 1;
    };
    auto rows_of = [&](int t) -> int { return t == p.nbi - 1 ? p.m_last : p.B; };
    auto issue_tile = [&](long long g0, unsigned nbuf) {      // one thread; the box is always 256 rows
        mbar_arrive_expect_tx(bar_full + 8 * nbuf, kXBytes);  // rows past n are zero-filled, still counted
        tma_load_2d(smem_u32(Xs) + nbuf * kXBytes, &tmapX, 0, (int)g0, bar_full + 8 * nbuf);
    };
    int t_cur = batch_index(0, 0);
    int t_next = total > 1 ? batch_index(1, 1 % p.nbi) : 0;
    seq = 2 % p.nbi;
    if (tid == 0) issue_tile((long long)t_cur * p.B, 0);

    const uint32_t taddr = tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + (warp >> 2) * 32;   // eq. 1 accumulators: columns 0-63
    const uint32_t tdw = tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + 64;                   // eq. 8 accumulator: columns 64-95
    float ycur = 0.f;
    {
        const long long r0 = (long long)t_cur * p.B;
        if (frow < min(BT, rows_of(t_cur))) ycur = __ldg(p.Y + r0 + frow);
    }
    const uint32_t ypp_a = smem_u32(ypp), yp_a = bar_yp;
    // instruction descriptors: D=f32, A=B=tf32, both K-major; eq. 1: M=128, N=32; eq. 8: M=64, N=32
    constexpr uint32_t idesc1 = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(S >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
    constexpr uint32_t idesc8 = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(kIn >> 3) << 17) | ((uint32_t)(64 >> 4) << 24);
    // position of (row r of the tile, column c) in the K-major operands of eq. 8: atom r/32, operand row c,
    // k = r%32 inside the 128-byte swizzled row
    const int ka = frow >> 5, kk = frow & 31;
    unsigned gt = 0;
    for (long long step = 0; step < total; ++step) {
        const int t_nn = (step + 2 < total) ? batch_index(step + 2, seq) : 0;
        seq = seq + 1 == p.nbi ? 0 : seq + 1;
        const long long r0 = (long long)t_cur * p.B;
        const int m = rows_of(t_cur);
        const int ntiles = (m + BT - 1) / BT;
        const float scale = t_cur == p.nbi - 1 ? p.scale_last : p.scale_full;   // eq. 5: 2 / m
        float g2 = 0.f;                                        // dW2 partial: unit lane, rows 32*warp.. of every tile

        for (int j = 0; j < ntiles; ++j, ++gt) {
            const unsigned buf = gt & 1u, ph = (gt >> 1) & 1u;
            const unsigned xst = gt % kRing, xph = (gt / kRing) & 1u;
            const int vt = min(BT, m - j * BT);
            long long nr0 = 0; int nrows = 0;
            if (j + 1 < ntiles) { nr0 = r0 + (long long)(j + 1) * BT; nrows = min(BT, m - (j + 1) * BT); }
            else if (step + 1 < total) { nr0 = (long long)t_next * p.B; nrows = min(BT, rows_of(t_next)); }
            if (warp == 0) {                                   // converged warp, one elected lane (uniform-register forms)
                if (elect_one()) {
                    mbar_arrive_expect_tx(bar_yp + 8 * buf, C * BT * 4);    // arm this tile's exchange
                    if (nrows > 0) {
                        const unsigned g1 = gt + 1, nbuf = g1 % kRing;
                        if (g1 >= kRing) mbar_wait(bar_empty + 8 * nbuf, ((g1 / kRing) - 1) & 1u);
                        issue_tile(nr0, nbuf);
                    }
                }
                __syncwarp();
            }
            float ynext = 0.f;
            if (frow < nrows) ynext = __ldg(p.Y + nr0 + frow);

            // ---------------- eq. 1 on the tensor cores ----------------
            mbar_wait(bar_full + 8 * xst, xph);
            const unsigned char* Xt_tile = Xs + xst * kXBytes;
            if (warp == 0) {
                tc_fence_after();
                if (elect_one()) {
                    const uint64_t bdesc = smem_desc_sw128(smem_u32(Wop));
#pragma unroll
                    for (int a = 0; a < 2; ++a) {              // rows 0-127 / 128-255 of the tile
                        const uint64_t adesc = smem_desc_sw128(smem_u32(Xs) + xst * kXBytes + a * 128 * 128);
#pragma unroll
                        for (int k = 0; k < kIn / 8; ++k)
                            mma_tf32(tmem_base + a * 32, adesc + 2 * k, bdesc + 2 * k, idesc1, k > 0);
                    }
                    tc_commit(bar_mma);
                }
                __syncwarp();
            }
            // while the MMA runs: this thread's X row, transposed into the B operand of eq. 8
            {
                float xr[kIn];
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    const float4 v = *reinterpret_cast<const float4*>(Xt_tile + swz(frow, c));
                    xr[4 * c] = v.x; xr[4 * c + 1] = v.y; xr[4 * c + 2] = v.z; xr[4 * c + 3] = v.w;
                }
#pragma unroll
                for (int i = 0; i < kIn; ++i)
                    *reinterpret_cast<float*>(Xt + ka * (32 * 128) + swz(i, kk >> 2) + (kk & 3) * 4) = xr[i];
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_empty + 8 * xst);   // this warp no longer reads the X tile
            mbar_wait(bar_mma, gt & 1u);
            tc_fence_after();
            float mk[kIn];                                     // ReLU'(z_u) w2_u of this row (eq. 7 factor, old W2)
            {
                uint32_t z[32];
                tmem_ld32(taddr, z);
                tmem_ld_wait();
                tc_fence_before();
                float pr[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    const float4 w = *reinterpret_cast<const float4*>(W2s + 4 * c);
                    float4 h;
                    h.x = fmaxf(__uint_as_float(z[4 * c]), 0.f);      h.y = fmaxf(__uint_as_float(z[4 * c + 1]), 0.f);   // eq. 2
                    h.z = fmaxf(__uint_as_float(z[4 * c + 2]), 0.f);  h.w = fmaxf(__uint_as_float(z[4 * c + 3]), 0.f);
                    *reinterpret_cast<float4*>(Hs + swz(frow, c)) = h;
                    mk[4 * c] = h.x > 0.f ? w.x : 0.f;     mk[4 * c + 1] = h.y > 0.f ? w.y : 0.f;
                    mk[4 * c + 2] = h.z > 0.f ? w.z : 0.f; mk[4 * c + 3] = h.w > 0.f ? w.w : 0.f;
                    pr[c & 3] = fmaf(h.x, w.x, fmaf(h.y, w.y, fmaf(h.z, w.z, fmaf(h.w, w.w, pr[c & 3]))));   // eq. 3
                }
                const float pv = (pr[0] + pr[1]) + (pr[2] + pr[3]);
#pragma unroll
                for (uint32_t dd = 0; dd < C; ++dd) {          // one hop to every CTA of the cluster
                    const uint32_t d = (crank + dd) & (C - 1);
                    st_async_f32(mapa(ypp_a + (buf * (C * BT) + crank * BT + frow) * 4, d), pv, mapa(yp_a + 8 * buf, d));
                }
            }
            // ---------------- eq. 5, eq. 7 ----------------
            mbar_wait(bar_yp + 8 * buf, ph);
            {
                const float* ypt = ypp + buf * (C * BT);
                float ypc[C];
#pragma unroll
                for (int c = 0; c < C; ++c) ypc[c] = ypt[c * BT + frow];
#pragma unroll
                for (int o = 1; o < C; o <<= 1)
#pragma unroll
                    for (int c = 0; c + o < C; c += 2 * o) ypc[c] += ypc[c + o];
                const float d = frow < vt ? scale * (ypc[0] - ycur) : 0.f;
                Ds[frow] = d;
#pragma unroll
                for (int u = 0; u < S; ++u)                    // dZ1^T[u][row]: A operand of eq. 8
                    *reinterpret_cast<float*>(At + ka * (64 * 128) + swz(u, kk >> 2) + (kk & 3) * 4) = d * mk[u];
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // At, Xt (generic writes) -> MMA
            __syncthreads();
            // ---------------- eq. 8 on the tensor cores: dW1^T += dZ1^T X ----------------
            if (warp == 0) {
                tc_fence_after();
                if (elect_one()) {
#pragma unroll
                    for (int a = 0; a < NA; ++a) {
                        const uint64_t adesc = smem_desc_sw128(smem_u32(At) + a * (64 * 128));
                        const uint64_t bdesc = smem_desc_sw128(smem_u32(Xt) + a * (32 * 128));
#pragma unroll
                        for (int k = 0; k < 4; ++k)
                            mma_tf32(tmem_base + 64, adesc + 2 * k, bdesc + 2 * k, idesc8, (j | a | k) != 0);
                    }
                    tc_commit(bar_mma2);
                }
                __syncwarp();
            }
            // meanwhile eq. 6 on the CUDA cores: unit = lane, rows 32*warp .. 32*warp+31 of the tile
            {
                float gp[4] = {0.f, 0.f, 0.f, 0.f};            // four independent chains hide the LDS latency
#pragma unroll
                for (int r = 0; r < 32; ++r) {
                    const int row = warp * 32 + r;
                    gp[r & 3] = fmaf(*reinterpret_cast<const float*>(Hs + swz(row, lane >> 2) + (lane & 3) * 4), Ds[row], gp[r & 3]);
                }
                g2 += (gp[0] + gp[1]) + (gp[2] + gp[3]);
            }
            ycur = ynext;
            mbar_wait(bar_mma2, gt & 1u);                      // eq. 8 of this tile has read At / Xt
            tc_fence_after();
            __syncthreads();                                   // and every warp is done with Hs / Ds
        }

        // ---------------- end of batch: eq. 9 ----------------
        part2[warp * S + lane] = g2;
        __syncthreads();
        if (warp < 2) {                                        // owners of the eq. 8 accumulator rows
            uint32_t dw[32];
            tmem_ld32(tdw, dw);
            tmem_ld_wait();
            tc_fence_before();
            if (wowner) {
#pragma unroll
                for (int i = 0; i < kIn; ++i) wrow[i] = fmaf(-p.lr, __uint_as_float(dw[i]), wrow[i]);   // W - lr*dW
                store_wop();
            }
        } else if (warp == 2) {                                // meanwhile eq. 9 for W2 (unit = lane)
            float sum = part2[lane];
#pragma unroll
            for (int w = 1; w < kWarps; ++w) sum += part2[w * S + lane];
            W2s[lane] -= p.lr * sum;
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");          // Wop -> next step's MMA
        __syncthreads();
        t_cur = t_next;
        t_next = t_nn;
    }

    // ---- write the trained slice back, free TMEM ---------------------------------------------------
    if (wowner) {
#pragma unroll
        for (int i = 0; i < kIn; ++i) p.W1[(size_t)i * H + crank * S + wu] = wrow[i];
    }
    if (tid < S) p.W2[crank * S + tid] = W2s[tid];
    if (crank == 0 && tid == 0 && p.stats) { p.stats[2] = (unsigned long long)total; p.stats[3] = C; p.stats[4] = bad_order; }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 128;" ::"r"(tmem_base) : "memory");
    }
    cluster_sync_all();        // no CTA exits while peers may still push into its shared memory
}

}  // namespace

bool train_tc_supported(int hidden, bool bf16) {
    if (bf16) return false;
    return hidden == 32 || hidden == 64 || hidden == 128 || hidden == 256;
}

cudaError_t launch_train_tc(const float* X, const float* Y, int64_t n, int batch, float lr, int epochs,
                            float* W1, float* W2, const int32_t* order, int hidden, bool bf16,
                            unsigned long long* stats, cudaStream_t stream, int64_t* launches) {
    if (!train_tc_supported(hidden, bf16) || n > 0x7fffffffLL - kBT) return cudaErrorInvalidValue;
    const int C = hidden / kS;
    TcParams p;
    p.Y = Y; p.n = n; p.B = batch; p.lr = lr;
    const long long nb = (n + batch - 1) / batch;
    p.total_steps = (long long)epochs * nb;
    p.nbi = (int)nb;
    p.m_last = (int)(n - (nb - 1) * batch);
    p.scale_full = 2.0f / (float)batch;
    p.scale_last = 2.0f / (float)p.m_last;
    p.W1 = W1; p.W2 = W2; p.order = order; p.H = hidden; p.stats = stats;
    if (p.total_steps == 0) return cudaSuccess;
    alignas(64) CUtensorMap tmap;
    if (!make_x_tensormap(&tmap, X, n, kBT)) return cudaErrorNotSupported;
    const size_t smem = (size_t)kRing * kXBytes + kS * 128 + (kBT / 32) * 64 * 128 + (kBT / 32) * 32 * 128 + kBT * 128 +
                        sizeof(float) * (2 * C * kBT + kWarps * kS + kS + kBT) + 8 * (2 * kRing + 4) + 16;
    auto launch = [&](auto kern) -> cudaError_t {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        if (C > 8) {
            e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
            if (e != cudaSuccess) return e;
        }
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(C);
        cfg.blockDim = dim3(kThreads);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = C;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        return cudaLaunchKernelEx(&cfg, kern, tmap, p);
    };
    cudaError_t err;
    switch (C) {
        case 1: err = launch(k_train_tf32<1>); break;
        case 2: err = launch(k_train_tf32<2>); break;
        case 4: err = launch(k_train_tf32<4>); break;
        case 8: err = launch(k_train_tf32<8>); break;
        default: return cudaErrorInvalidValue;
    }
    if (err == cudaSuccess) ++*launches;
    return err;
}

}  // namespace mlp
