// train_tf32.cu -- tensor-core variant of the fused training kernel (SURVEY.md 8(a) row a-T,
// 8(f) NEXT-2; BASELINE.json: "allowed only as a separately reported variant with its own stated
// tolerance").  Same method, same loop, same cluster layout as train_fused.cu (eqs. 1-9,
// PAPER.md:44-71; one launch for every batch of every epoch), but eq. 1 (Z1 = X W1) runs on the
// tensor cores: per 256-row tile two tcgen05.mma chains (M=128, N=32 hidden units of this CTA,
// K=32 in four K=8 steps, kind::tf32: fp32 operands truncated to TF32, fp32 accumulate in TMEM).
// Everything else stays fp32 on the CUDA cores.  Hidden 256 on a cluster of 8 CTAs only.
//
// Per tile and CTA (8 warps):
//   TMA (cp.async.bulk.tensor, 128-byte swizzle) brings the X tile [256 x 32] one tile ahead;
//   warp 0 issues the 8 MMAs (A = X tile, B = W1 slice kept in shared memory in operand layout);
//   every thread owns ONE row: it reads its 32 pre-activations from TMEM (tcgen05.ld), applies
//   eq. 2, stores H to shared memory, forms its partial of eq. 3 and pushes it to the 8 CTAs
//   (st.async + mbarrier, as in train_fused.cu); after the exchange it computes dZ2 (eq. 5);
//   the backward pass (eqs. 6-8) is the K-split FFMA2 loop of train_fused.cu reading H and dZ2
//   from shared memory; per-warp partials, fixed-order cross-warp sum and eq. 9 as there, with
//   the updated W1 written both to the fp32 master copy and to the MMA operand layout.
// No W1 register file, hence no reload between steps.
#include <cuda.h>

#include "common.cuh"
#include "internal.h"

namespace mlp {
namespace {

constexpr int kS = 32;            // hidden units per CTA
constexpr int kC = 8;             // cluster size
constexpr int kBT = 256;          // rows per tile
constexpr int kWarps = 8;
constexpr int kThreads = kWarps * 32;
constexpr int kRing = 3;          // X ring stages
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
};

__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* tmap, int c0, int c1, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
        ::"r"(dst), "l"(tmap), "r"(c0), "r"(c1), "r"(bar)
        : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mma_tf32(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                         uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]),
          "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]),
          "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]),
          "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ bool elect_one() {
    uint32_t pred = 0;
    asm volatile("{\n\t.reg .pred P;\n\telect.sync _|P, 0xffffffff;\n\tselp.u32 %0, 1, 0, P;\n\t}" : "=r"(pred));
    return pred != 0;
}
// K-major, 128-byte-swizzled operand descriptor (8-row x 128-byte atoms, 1024 bytes apart)
__device__ __forceinline__ uint64_t smem_desc_sw128(uint32_t saddr) {
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | (1ull << 16) | (64ull << 32) | (1ull << 46) | (2ull << 61);
}
// The gradient partials and the fp32 master copy keep hidden unit u in slot (u % 4) * 8 + u / 4, so that the
// lanes of a sub-group (units 4*lu + j) store to consecutive 16-byte slots (no bank conflicts).
__device__ __forceinline__ int unit_of(int sl) { return (sl & 7) * 4 + (sl >> 3); }
// byte offset of the 16-byte chunk c of row r in a [rows][128 B] tile with the 128-byte swizzle
__device__ __forceinline__ int swz(int r, int c) { return r * 128 + ((c ^ (r & 7)) << 4); }

__global__ void __launch_bounds__(kThreads, 1)
k_train_tf32(const __grid_constant__ CUtensorMap tmapX, const TcParams p) {
    constexpr int S = kS, BT = kBT, C = kC;
    constexpr int LPS = 8, SPW = 4, RB = BT / SPW, ITER = RB / kWarps;   // backward mapping (train_fused.cu)
    constexpr int IPS = kIn / SPW;                                        // inputs per sub-group
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char* Xs = smem;                                             // [kRing][32 KB] swizzled rows
    unsigned char* Wop = Xs + kRing * kXBytes;                            // [S][128 B] B operand (K-major, swizzled)
    unsigned char* Hs = Wop + S * 128;                                    // [BT][128 B] H = ReLU(Z1), swizzled rows
    unsigned char* Ms = Hs + BT * 128;                                    // [BT][128 B] ReLU'(Z1) * W2 (eq. 7 factor), swizzled
    float* part = reinterpret_cast<float*>(Ms + BT * 128);                // [kWarps][S*32]  layout [q][slot][4]
    float* W1m = part + kWarps * S * kIn;                                 // [S*32] fp32 master, layout [q][slot][4]
    float* ypp = W1m + S * kIn;                                           // [2][C][BT]
    float* part2 = ypp + 2 * C * BT;                                      // [kWarps][S]
    float* W2s = part2 + kWarps * S;                                      // [S]
    float* Ds = W2s + S;                                                  // [BT] dZ2 of the tile
    uint64_t* bars = reinterpret_cast<uint64_t*>(Ds + BT);                // full[3], empty[3], yp[2], mma
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * kRing + 3);
    const uint32_t bar_full = smem_u32(bars), bar_empty = smem_u32(bars + kRing),
                   bar_yp = smem_u32(bars + 2 * kRing), bar_mma = smem_u32(bars + 2 * kRing + 2);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int lu = lane % LPS, s = lane / LPS;
    const uint32_t crank = cluster_ctarank();
    const int H = p.H;

    // ---- one-time setup ---------------------------------------------------------------------------
    for (int f = tid; f < S * kIn; f += kThreads) {
        const int q = f / (S * 4), rem = f % (S * 4), u = unit_of(rem >> 2), r = rem & 3, i = q * 4 + r;
        const float w = p.W1[(size_t)i * H + crank * S + u];
        W1m[f] = w;
        *reinterpret_cast<float*>(Wop + swz(u, q) + r * 4) = w;           // B[n = u][k = i]
    }
    if (tid < S) W2s[tid] = p.W2[crank * S + tid];
    if (tid == 0) {
        for (int b = 0; b < kRing; ++b) { mbar_init(bar_full + 8 * b, 1); mbar_init(bar_empty + 8 * b, kWarps); }
        mbar_init(bar_yp, 1); mbar_init(bar_yp + 8, 1); mbar_init(bar_mma, 1);
        fence_mbar_init();
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 64;" ::"r"(smem_u32(tmem_slot)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");          // Wop (generic writes) -> MMA (async proxy)
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    if (smem_u32(smem) & 1023u) __trap();
    cluster_sync_all();        // every CTA's barriers exist before anyone pushes to them

    const long long total = p.total_steps;
    int seq = 0;
    auto batch_index = [&](long long step, int sq) -> int { return p.order ? __ldg(p.order + step) : sq; };
    auto rows_of = [&](int t) -> int { return t == p.nbi - 1 ? p.m_last : p.B; };
    auto issue_tile = [&](long long g0, unsigned nbuf) {      // one thread; the box is always 256 rows
        mbar_arrive_expect_tx(bar_full + 8 * nbuf, kXBytes);  // rows past n are zero-filled, still counted
        tma_load_2d(smem_u32(Xs) + nbuf * kXBytes, &tmapX, 0, (int)g0, bar_full + 8 * nbuf);
    };
    int t_cur = batch_index(0, 0);
    int t_next = total > 1 ? batch_index(1, 1 % p.nbi) : 0;
    seq = 2 % p.nbi;
    if (tid == 0) issue_tile((long long)t_cur * p.B, 0);

    // forward ownership: thread <-> tile row (TMEM lane rule: warp w reads lanes 32*(w%4)..)
    const int frow = (warp >> 2) * 128 + (warp & 3) * 32 + lane;
    const uint32_t taddr = tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + (warp >> 2) * 32;
    float ycur = 0.f;
    {
        const long long r0 = (long long)t_cur * p.B;
        if (frow < min(BT, rows_of(t_cur))) ycur = __ldg(p.Y + r0 + frow);
    }
    // Ypred exchange: peer CTA addresses
    const uint32_t ypp_a = smem_u32(ypp), yp_a = bar_yp;
    const int rowl = warp * ITER;
    float* mypart = part + warp * (S * kIn);

    constexpr uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(S >> 3) << 17) |
                               ((uint32_t)(128 >> 4) << 24);
    unsigned gt = 0;
    for (long long step = 0; step < total; ++step) {
        const int t_nn = (step + 2 < total) ? batch_index(step + 2, seq) : 0;
        seq = seq + 1 == p.nbi ? 0 : seq + 1;
        const long long r0 = (long long)t_cur * p.B;
        const int m = rows_of(t_cur);
        const int ntiles = (m + BT - 1) / BT;
        const float scale = t_cur == p.nbi - 1 ? p.scale_last : p.scale_full;   // eq. 5: 2 / m
        float g2[4] = {0.f, 0.f, 0.f, 0.f};

        for (int j = 0; j < ntiles; ++j, ++gt) {
            const unsigned buf = gt & 1u, ph = (gt >> 1) & 1u;
            const unsigned xst = gt % kRing, xph = (gt / kRing) & 1u;
            const int vt = min(BT, m - j * BT);
            long long nr0 = 0; int nrows = 0;
            if (j + 1 < ntiles) { nr0 = r0 + (long long)(j + 1) * BT; nrows = min(BT, m - (j + 1) * BT); }
            else if (step + 1 < total) { nr0 = (long long)t_next * p.B; nrows = min(BT, rows_of(t_next)); }
            if (tid == 0) {
                mbar_arrive_expect_tx(bar_yp + 8 * buf, C * BT * 4);        // arm this tile's exchange
                if (nrows > 0) {
                    const unsigned g1 = gt + 1, nbuf = g1 % kRing;
                    if (g1 >= kRing) mbar_wait(bar_empty + 8 * nbuf, ((g1 / kRing) - 1) & 1u);
                    issue_tile(nr0, nbuf);
                }
            }
            __syncwarp();
            float ynext = 0.f;
            if (frow < nrows) ynext = __ldg(p.Y + nr0 + frow);

            // ---------------- forward: eq. 1 on the tensor cores ----------------
            mbar_wait(bar_full + 8 * xst, xph);                // every warp reads X later (backward)
            if (warp == 0) {
                tc_fence_after();
                if (elect_one()) {
                    const uint64_t bdesc = smem_desc_sw128(smem_u32(Wop));
#pragma unroll
                    for (int a = 0; a < 2; ++a) {              // rows 0-127 / 128-255 of the tile
                        const uint64_t adesc = smem_desc_sw128(smem_u32(Xs) + xst * kXBytes + a * 128 * 128);
#pragma unroll
                        for (int k = 0; k < kIn / 8; ++k)
                            mma_tf32(tmem_base + a * 32, adesc + 2 * k, bdesc + 2 * k, idesc, k > 0);
                    }
                    tc_commit(bar_mma);
                }
                __syncwarp();
            }
            mbar_wait(bar_mma, gt & 1u);
            tc_fence_after();
            __syncthreads();                                   // every warp is done with H / dZ2 of the previous tile
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
                    *reinterpret_cast<float4*>(Ms + swz(frow, c)) =                       // eq. 7: ReLU'(z) w2 (old W2)
                        make_float4(h.x > 0.f ? w.x : 0.f, h.y > 0.f ? w.y : 0.f, h.z > 0.f ? w.z : 0.f, h.w > 0.f ? w.w : 0.f);
                    pr[c & 3] = fmaf(h.x, w.x, fmaf(h.y, w.y, fmaf(h.z, w.z, fmaf(h.w, w.w, pr[c & 3]))));   // eq. 3
                }
                const float pv = (pr[0] + pr[1]) + (pr[2] + pr[3]);
#pragma unroll
                for (uint32_t dd = 0; dd < C; ++dd) {          // one hop to every CTA of the cluster
                    const uint32_t d = (crank + dd) & (C - 1);
                    st_async_f32(mapa(ypp_a + (buf * (C * BT) + crank * BT + frow) * 4, d), pv, mapa(yp_a + 8 * buf, d));
                }
            }
            // ---------------- eq. 5 ----------------
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
                Ds[frow] = frow < vt ? scale * (ypc[0] - ycur) : 0.f;
            }
            __syncthreads();                                   // H and dZ2 of the whole tile are in shared memory

            // ---------------- backward: eqs. 6-8, K-split over the sub-groups ----------------
            // lane (s, lu): units 4*lu..4*lu+3, inputs [IPS*s, IPS*(s+1)), rows of ALL sub-groups
            const unsigned char* Xt = Xs + xst * kXBytes;
            f32x2 acc[4][IPS / 2];
#pragma unroll
            for (int it = 0; it < ITER; ++it) {
#pragma unroll
                for (int t = 0; t < SPW; ++t) {
                    const int r = (s ^ t) * RB + rowl + it;                    // tile row
                    const float d = Ds[r];
                    const float4 mk = *reinterpret_cast<const float4*>(Ms + swz(r, lu));
                    const float mm[4] = {mk.x, mk.y, mk.z, mk.w};
                    if (t == 0) {                                              // eq. 6 (each row once per CTA)
                        const float4 h = *reinterpret_cast<const float4*>(Hs + swz(r, lu));
                        g2[0] = fmaf(h.x, d, g2[0]); g2[1] = fmaf(h.y, d, g2[1]);
                        g2[2] = fmaf(h.z, d, g2[2]); g2[3] = fmaf(h.w, d, g2[3]);
                    }
                    f32x2 dd[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const float e = d * mm[u];                             // eq. 7
                        dd[u] = pack2(e, e);
                    }
#pragma unroll
                    for (int x = 0; x < IPS / 4; ++x) {                        // eq. 8
                        const ulonglong2 xv = *reinterpret_cast<const ulonglong2*>(Xt + swz(r, (IPS / 4) * s + x));
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            if (it == 0 && t == 0) {
                                acc[u][2 * x] = fmul2(xv.x, dd[u]);
                                acc[u][2 * x + 1] = fmul2(xv.y, dd[u]);
                            } else {
                                ffma2(acc[u][2 * x], xv.x, dd[u]);
                                ffma2(acc[u][2 * x + 1], xv.y, dd[u]);
                            }
                        }
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_empty + 8 * xst);   // this warp is done with the X tile
            ycur = ynext;
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int x = 0; x < IPS / 4; ++x) {
                    const int q = (IPS / 4) * s + x;
                    ulonglong2* dst = reinterpret_cast<ulonglong2*>(mypart + (q * S + u * 8 + lu) * 4);   // slot_of(4*lu+u)
                    f32x2 lo = acc[u][2 * x], hi = acc[u][2 * x + 1];
                    if (j > 0) {                               // later tiles of a large batch
                        const ulonglong2 old = *dst;
                        lo = fadd2(lo, old.x); hi = fadd2(hi, old.y);
                    }
                    *dst = make_ulonglong2(lo, hi);
                }
        }

        // ---------------- end of batch: reduce partial gradients, eq. 9 ----------------
#pragma unroll
        for (int o = LPS; o < 32; o <<= 1)
#pragma unroll
            for (int u = 0; u < 4; ++u) g2[u] += __shfl_xor_sync(0xffffffffu, g2[u], o);
        if (s == 0) {
#pragma unroll
            for (int u = 0; u < 4; ++u) part2[warp * S + 4 * lu + u] = g2[u];
        }
        __syncthreads();
        {
            constexpr int NF = S * 8;                          // float4 slots of this CTA's dW1 (= kThreads)
            const f32x2 nlr2 = pack2(-p.lr, -p.lr);
            const int f = tid;
            ulonglong2 v[kWarps];
#pragma unroll
            for (int w = 0; w < kWarps; ++w) v[w] = reinterpret_cast<const ulonglong2*>(part)[w * NF + f];
#pragma unroll
            for (int o = 1; o < kWarps; o <<= 1)               // fixed pairwise tree over warps
#pragma unroll
                for (int w = 0; w + o < kWarps; w += 2 * o) {
                    v[w].x = fadd2(v[w].x, v[w + o].x);
                    v[w].y = fadd2(v[w].y, v[w + o].y);
                }
            ulonglong2 wv = reinterpret_cast<ulonglong2*>(W1m)[f];
            ffma2(wv.x, v[0].x, nlr2);                                         // eq. 9: W - lr*dW
            ffma2(wv.y, v[0].y, nlr2);
            reinterpret_cast<ulonglong2*>(W1m)[f] = wv;
            const int q = f / S, u = unit_of(f % S);          // same float4 in the MMA operand layout
            *reinterpret_cast<ulonglong2*>(Wop + swz(u, q)) = wv;
        }
        if (tid < S) {
            float sum = part2[tid];
#pragma unroll
            for (int w = 1; w < kWarps; ++w) sum += part2[w * S + tid];
            W2s[tid] -= p.lr * sum;                                            // eq. 9
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");          // Wop -> next step's MMA
        __syncthreads();
        t_cur = t_next;
        t_next = t_nn;
    }

    // ---- write the trained slice back, free TMEM ---------------------------------------------------
    for (int f = tid; f < S * kIn; f += kThreads) {
        const int q = f / (S * 4), rem = f % (S * 4), u = unit_of(rem >> 2), i = q * 4 + (rem & 3);
        p.W1[(size_t)i * H + crank * S + u] = W1m[f];
    }
    if (tid < S) p.W2[crank * S + tid] = W2s[tid];
    tc_fence_before();
    __syncthreads();
    if (warp == 0) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 64;" ::"r"(tmem_base) : "memory");
    }
    cluster_sync_all();        // no CTA exits while peers may still push into its shared memory
}

}  // namespace

bool train_tf32_supported(int hidden) { return hidden == kS * kC; }

cudaError_t launch_train_tf32(const float* X, const float* Y, int64_t n, int batch, float lr, int epochs,
                              float* W1, float* W2, const int32_t* order, int hidden,
                              cudaStream_t stream, int64_t* launches) {
    if (hidden != kS * kC || n > 0x7fffffffLL - kBT) return cudaErrorInvalidValue;
    TcParams p;
    p.Y = Y; p.n = n; p.B = batch; p.lr = lr;
    const long long nb = (n + batch - 1) / batch;
    p.total_steps = (long long)epochs * nb;
    p.nbi = (int)nb;
    p.m_last = (int)(n - (nb - 1) * batch);
    p.scale_full = 2.0f / (float)batch;
    p.scale_last = 2.0f / (float)p.m_last;
    p.W1 = W1; p.W2 = W2; p.order = order; p.H = hidden;
    if (p.total_steps == 0) return cudaSuccess;
    alignas(64) CUtensorMap tmap;
    if (!make_x_tensormap(&tmap, X, n, kBT)) return cudaErrorNotSupported;
    const size_t smem = (size_t)kRing * kXBytes + kS * 128 + 2 * kBT * 128 +
                        sizeof(float) * (kWarps * kS * kIn + kS * kIn + 2 * kC * kBT + kWarps * kS + kS + kBT) +
                        8 * (2 * kRing + 3) + 16;
    cudaError_t err = cudaFuncSetAttribute(k_train_tf32, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err != cudaSuccess) return err;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(kC);
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = kC;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    err = cudaLaunchKernelEx(&cfg, k_train_tf32, tmap, p);
    if (err == cudaSuccess) ++*launches;
    return err;
}

}  // namespace mlp
