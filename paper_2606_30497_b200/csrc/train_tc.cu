// train_tc.cu -- tensor-core variants of the fused training kernel (SURVEY.md 8(a) row a-T, 8(f) NEXT-2;
// BASELINE.json: "allowed only as a separately reported variant with its own stated tolerance").
// Same method, same loop, same cluster layout and Ypred exchange as train_fused.cu (eqs. 1-9,
// PAPER.md:44-71; one launch for every batch of every epoch), but both large products run on the
// tensor cores (tcgen05.mma, fp32 accumulate in TMEM, fp32 master weights):
//   eq. 1  Z1 = X W1        per tile chains of M=128 (rows), N=32 or 64 (units of this CTA), K=32;
//   eq. 8  dW1^T = dZ1^T X  one chain M=64 (units), N=32 (inputs), K = rows of the tile, accumulated in
//                           TMEM across the tiles of a batch.  TF32 with 32 units per CTA: the two row halves
//                           of the tile run side by side (M=64 = units x 2 halves, N=64 = inputs x 2 halves,
//                           half as many MMAs) and the two diagonal blocks are summed at the end of the batch.
// Operand precision: TF32 (kind::tf32: fp32 bits in shared memory, truncated by the tensor core) or BF16
// (kind::f16: the threads round every operand to BF16, round to nearest even, as they stage it).
// Everything else stays fp32 on the CUDA cores.
//
// Two geometries (template parameter S = hidden units per CTA):
//   S = 32: 256-row tiles, a thread owns ONE row;        hidden 32..256  on clusters of 1..8 CTAs,
//   S = 64: 128-row tiles, TWO threads share a row (32 units each); hidden 512, 1024 on clusters of 8, 16.
//
// Per tile and CTA (8 warps):
//   TMA (cp.async.bulk.tensor, 128-byte swizzle) brings the X tile one tile ahead; warp 0 issues eq. 1
//   (A = X tile, B = W1^T slice in operand layout); meanwhile every thread transposes its part of its X
//   row into the K-major B operand of eq. 8; then it reads its 32 pre-activations from TMEM, applies
//   eq. 2, stores H, forms its partial of eq. 3 and pushes it to every CTA of the cluster (st.async +
//   mbarrier); after the exchange it computes dZ2 (eq. 5) and writes its part of dZ1 = dZ2 ReLU'(Z1) W2
//   (eq. 7) into the K-major A operand of eq. 8; warp 0 issues eq. 8 while all warps do eq. 6 (dW2) on
//   the CUDA cores.  At the end of the batch the threads that own the TMEM rows of dW1^T (one per hidden
//   unit) apply eq. 9 to the fp32 master row they keep in registers and rewrite their row of the eq. 1
//   operand.  BF16 mode: all operands K-major with the 128-byte swizzle (the conventions of eval_tc.cu), the two
//   operands of eq. 8 transposed by the threads with 2-byte stores.  TF32 mode: the X tile arrives with the
//   32-byte-atom flavour of the 128-byte swizzle, in which a TF32 operand can be read K-major (eq. 1) AND MN-major
//   (tc_common.cuh): eq. 8 takes the tile itself as its B operand and dZ1 as the threads produce it (a row = 32
//   units = 128 bytes) as its A operand: no transposing stores, the threads never read X.
#include <cuda.h>

#include "tc_common.cuh"

namespace mlp {
namespace {

constexpr int kWarps = 8;
constexpr int kThreads = kWarps * 32;
constexpr int kRing = 2;          // X ring stages

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

// shared-memory plan, shared by the kernel and its launcher
template <int C, int S, bool BF16>
struct TcPlan {
    static constexpr int NTH = S / 32;                 // threads per row
    static constexpr int BT = 256 / NTH;               // rows per tile
    static constexpr int NSL = C * NTH;                // Ypred partial slots per row
    static constexpr uint32_t XBYTES = BT * 128;       // one X tile
    static constexpr uint32_t oX = 0;                                   // [kRing][BT][128 B]  A of eq. 1 (TF32)
    static constexpr uint32_t oXb = oX + kRing * XBYTES;                // [BT][128 B]         A of eq. 1 (BF16 copy)
    static constexpr uint32_t oW = oXb + (BF16 ? XBYTES : 0);           // [S][128 B]          B of eq. 1
    static constexpr uint32_t oAt = oW + S * 128;                       // A of eq. 8 (dZ1 rows, MN-major): BF16 [BT][64 units x 2 B]; TF32 [2 planes][BT][32 units x 4 B]
    static constexpr uint32_t oXt = oAt + (BF16 ? BT * 128 : BT * 256);                     // (end of At; B of eq. 8 is the X tile itself, MN-major: the BF16 copy or the landed TF32 tile)
    static constexpr uint32_t oH = oXt;                                 // [NTH][BT][128 B]    H = ReLU(Z1)
    static constexpr uint32_t oYp = oH + NTH * BT * 128;                // [2][NSL][BT] floats
    static constexpr uint32_t oP2 = oYp + 2 * NSL * BT * 4;             // [kWarps][32] dW2 partials
    static constexpr uint32_t oW2 = oP2 + kWarps * 32 * 4;              // [S]
    static constexpr uint32_t oD = oW2 + S * 4;                         // [BT] dZ2 of the tile
    static constexpr uint32_t oBar = (oD + BT * 4 + 7) / 8 * 8;         // full[kRing], empty[kRing], yp[2], mma, mma2
    static constexpr uint32_t oTm = oBar + 8 * (2 * kRing + 4);
    static constexpr uint32_t BYTES = oTm + 16;
};

// 8 floats -> 8 packed bf16 (16 bytes)
__device__ __forceinline__ uint4 pack_bf16x8(const float* v) {
    return make_uint4(bf16x2(v[0], v[1]), bf16x2(v[2], v[3]), bf16x2(v[4], v[5]), bf16x2(v[6], v[7]));
}

template <int C, int S, bool BF16>
__global__ void __launch_bounds__(kThreads, 1)
k_train_tc(const __grid_constant__ CUtensorMap tmapX, const TcParams p) {
    using P = TcPlan<C, S, BF16>;
    constexpr int NTH = P::NTH, BT = P::BT, NSL = P::NSL;
    constexpr uint32_t kXBytes = P::XBYTES;
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char* Xs = smem + P::oX;
    unsigned char* Xb = smem + P::oXb;
    unsigned char* Wop = smem + P::oW;
    unsigned char* At = smem + P::oAt;
    unsigned char* Hs = smem + P::oH;
    float* ypp = reinterpret_cast<float*>(smem + P::oYp);
    float* part2 = reinterpret_cast<float*>(smem + P::oP2);
    float* W2s = reinterpret_cast<float*>(smem + P::oW2);
    float* Ds = reinterpret_cast<float*>(smem + P::oD);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + P::oBar);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + P::oTm);
    const uint32_t bar_full = smem_u32(bars), bar_empty = smem_u32(bars + kRing),
                   bar_yp = smem_u32(bars + 2 * kRing), bar_mma = smem_u32(bars + 2 * kRing + 2),
                   bar_mma2 = smem_u32(bars + 2 * kRing + 3);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t crank = cluster_ctarank();
    const int H = p.H;
    // thread <-> (tile row, 32-unit half); TMEM lane rule: warp w reads lanes 32*(w%4)..
    const int blk = warp >> 2, wq = warp & 3;
    const int frow = (NTH == 1 ? blk * 128 : 0) + wq * 32 + lane;
    const int hb = NTH == 2 ? blk : 0;                                    // which 32 of the CTA's S units
    const int uoff = hb * 32;
    // weight ownership: the M=64 accumulator of eq. 8 keeps unit u in TMEM lane (u/16)*32 + u%16, i.e. lanes
    // 0-15 of warps 0..S/16-1: those threads hold the fp32 master row W1[:, u] in registers for the whole run
    const bool wowner = warp < S / 16 && lane < 16;
    const int wu = warp * 16 + lane;                                      // owned hidden unit (if wowner)
    float wrow[kIn];
#pragma unroll
    for (int i = 0; i < kIn; ++i) wrow[i] = wowner ? p.W1[(size_t)i * H + crank * S + wu] : 0.f;
    auto store_wop = [&]() {                                              // B[n = u][k = i], eq. 1 operand
        if constexpr (BF16) {
#pragma unroll
            for (int c = 0; c < 4; ++c) *reinterpret_cast<uint4*>(Wop + swz(wu, c)) = pack_bf16x8(wrow + 8 * c);
        } else {
#pragma unroll
            for (int c = 0; c < 8; ++c)
                *reinterpret_cast<float4*>(Wop + swz(wu, c)) = make_float4(wrow[4 * c], wrow[4 * c + 1], wrow[4 * c + 2], wrow[4 * c + 3]);
        }
    };

    // ---- one-time setup ---------------------------------------------------------------------------
    if (wowner) store_wop();
    for (int f = tid; f < (int)(P::oXt - P::oAt) / 4; f += kThreads) reinterpret_cast<float*>(At)[f] = 0.f;   // padding rows / plane stay 0
    if constexpr (BF16)                                                   // the unused half of every row of the BF16 tile copy (read as N = 32..63 by eq. 8)
        for (int f = tid; f < BT * 32; f += kThreads) reinterpret_cast<float*>(Xb)[f] = 0.f;
    if (tid < S) W2s[tid] = p.W2[crank * S + tid];
    if (tid == 0) {
        for (int b = 0; b < kRing; ++b) { mbar_init(bar_full + 8 * b, 1); mbar_init(bar_empty + 8 * b, BF16 ? kWarps : 1); }
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
    // The table entry of step k is loaded when step k-3 starts and only looked at (range check) when step k-2
    // starts, so the global-load latency never sits on a step's critical path (as in train_fused.cu).
    auto checked = [&](int t, int sq) -> int {
        if (!p.order) return sq;
        if ((unsigned)t < (unsigned)p.nbi) return t;
        ++bad_order;
        return t < 0 ? 0 : p.nbi - 1;
    };
    auto raw_entry = [&](long long step) -> int { return (p.order && step < total) ? __ldg(p.order + step) : 0; };
    auto rows_of = [&](int t) -> int { return t == p.nbi - 1 ? p.m_last : p.B; };
    auto issue_tile = [&](long long g0, unsigned nbuf) {      // one thread; the box is always BT rows
        mbar_arrive_expect_tx(bar_full + 8 * nbuf, kXBytes);  // rows past n are zero-filled, still counted
        tma_load_2d(smem_u32(Xs) + nbuf * kXBytes, &tmapX, 0, (int)g0, bar_full + 8 * nbuf);
    };
    int t_cur = checked(raw_entry(0), 0);
    int t_next = total > 1 ? checked(raw_entry(1), 1 % p.nbi) : 0;
    int raw2 = raw_entry(2);                          // entry of step + 2, not yet checked
    seq = 2 % p.nbi;
    if (tid == 0) issue_tile((long long)t_cur * p.B, 0);

    const uint32_t taddr = tmem_base + ((uint32_t)(wq * 32) << 16) + blk * 32;   // eq. 1 accumulators: columns 0-63
    const uint32_t tdw = tmem_base + ((uint32_t)(wq * 32) << 16) + 64;           // eq. 8 accumulator: columns 64-95
    float ycur = 0.f;
    {
        const long long r0 = (long long)t_cur * p.B;
        if (frow < min(BT, rows_of(t_cur))) ycur = __ldg(p.Y + r0 + frow);
    }
    const uint32_t ypp_a = smem_u32(ypp), yp_a = bar_yp;
    // instruction descriptors: D=f32, both operands K-major; eq. 1: M=128, N=32 (two chains) or 64; eq. 8: M=64, N=32
    constexpr uint32_t kFmt = BF16 ? 1u : 2u;
    constexpr uint32_t idesc1 = mma_idesc(kFmt, 128, S == 32 ? 32 : 64);
    constexpr uint32_t idesc8 = mma_idesc(kFmt, 64, kIn);
    // TF32, 32 units per CTA (one thread per tile row, BT = 256): eq. 8 folds the tile's two row halves side by side
    // (see there), 16 MMAs of N = 64 instead of 32 of N = 32
    constexpr bool FOLD = !BF16 && S == 32;
    constexpr uint32_t idesc8f = mma_idesc(kFmt, 64, 2 * kIn);
    constexpr int KS1 = BF16 ? 2 : 4;                          // MMAs per chain of eq. 1 (K = 16 or 8 each)
    constexpr int NCH = 8 / NTH;                               // 16-byte chunks of an X row this thread handles
    const int c0 = NTH == 2 ? hb * 4 : 0;
    unsigned gt = 0;
    for (long long step = 0; step < total; ++step) {
        const int t_nn = (step + 2 < total) ? checked(raw2, seq) : 0;
        raw2 = raw_entry(step + 3);
        seq = seq + 1 == p.nbi ? 0 : seq + 1;
        const long long r0 = (long long)t_cur * p.B;
        const int m = rows_of(t_cur);
        const int ntiles = (m + BT - 1) / BT;
        const float scale = t_cur == p.nbi - 1 ? p.scale_last : p.scale_full;   // eq. 5: 2 / m
        float g2 = 0.f;                                        // dW2 partial of one unit over 32 rows of every tile

        for (int j = 0; j < ntiles; ++j, ++gt) {
            const unsigned buf = gt & 1u, ph = (gt >> 1) & 1u;
            const unsigned xst = gt % kRing, xph = (gt / kRing) & 1u;
            const int vt = min(BT, m - j * BT);
            long long nr0 = 0; int nrows = 0;
            if (j + 1 < ntiles) { nr0 = r0 + (long long)(j + 1) * BT; nrows = min(BT, m - (j + 1) * BT); }
            else if (step + 1 < total) { nr0 = (long long)t_next * p.B; nrows = min(BT, rows_of(t_next)); }
            if (warp == 0) {                                   // converged warp, one elected lane (uniform-register forms)
                if (elect_one()) {
                    mbar_arrive_expect_tx(bar_yp + 8 * buf, NSL * BT * 4);  // arm this tile's exchange
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
            const unsigned char* Xtile = Xs + xst * kXBytes;
            auto issue_eq1 = [&]() {
                if (warp == 0) {
                    tc_fence_after();
                    if (elect_one()) {
                        const uint64_t bdesc = smem_desc_sw128(smem_u32(Wop));
#pragma unroll
                        for (int a = 0; a < (NTH == 1 ? 2 : 1); ++a) {     // row blocks of 128 (S = 32: two of them)
                            const uint64_t adesc = BF16 ? smem_desc_sw128(smem_u32(Xb) + a * 128 * 128)
                                                        : smem_desc_sw128_a32(smem_u32(Xs) + xst * kXBytes + a * 128 * 128, 1024);
#pragma unroll
                            for (int k = 0; k < KS1; ++k) {
                                if constexpr (BF16) mma_f16(tmem_base + a * 32, adesc + 2 * k, bdesc + 2 * k, idesc1, k > 0);
                                else mma_tf32(tmem_base + a * 32, adesc + 2 * k, bdesc + 2 * k, idesc1, k > 0);
                            }
                        }
                        tc_commit(bar_mma);
                    }
                    __syncwarp();
                }
            };
            if constexpr (!BF16) issue_eq1();                  // TF32: the tile is the operand as TMA delivered it
            // BF16: this thread's part of its X row, rounded into the BF16 copy of the tile (A of eq. 1 K-major, B of eq. 8 MN-major)
            // (TF32: the tile is read by the tensor core only, in both orientations; eq. 8's commit releases the slot)
            if constexpr (BF16) {
                float xr[4 * NCH];
#pragma unroll
                for (int c = 0; c < NCH; ++c) {
                    const float4 v = *reinterpret_cast<const float4*>(Xtile + swz(frow, c0 + c));
                    xr[4 * c] = v.x; xr[4 * c + 1] = v.y; xr[4 * c + 2] = v.z; xr[4 * c + 3] = v.w;
                }
#pragma unroll
                for (int c = 0; c < NCH / 2; ++c)          // 16-byte chunk c0/2 + c holds inputs 8 (c0/2 + c) .. + 7
                    *reinterpret_cast<uint4*>(Xb + swz(frow, c0 / 2 + c)) = pack_bf16x8(xr + 8 * c);
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                __syncthreads();                           // every row of the BF16 copy is written
                issue_eq1();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_empty + 8 * xst);   // this warp no longer reads the X tile
            }
            mbar_wait(bar_mma, gt & 1u);
            tc_fence_after();
            float mk[32];                                      // ReLU'(z_u) w2_u of this row (eq. 7 factor, old W2)
            {
                uint32_t z[32];
                tmem_ld32(taddr, z);
                tmem_ld_wait();
                tc_fence_before();
                float pr[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    const float4 w = *reinterpret_cast<const float4*>(W2s + uoff + 4 * c);
                    float4 h;
                    h.x = fmaxf(__uint_as_float(z[4 * c]), 0.f);      h.y = fmaxf(__uint_as_float(z[4 * c + 1]), 0.f);   // eq. 2
                    h.z = fmaxf(__uint_as_float(z[4 * c + 2]), 0.f);  h.w = fmaxf(__uint_as_float(z[4 * c + 3]), 0.f);
                    *reinterpret_cast<float4*>(Hs + hb * (BT * 128) + swz(frow, c)) = h;
                    mk[4 * c] = h.x > 0.f ? w.x : 0.f;     mk[4 * c + 1] = h.y > 0.f ? w.y : 0.f;
                    mk[4 * c + 2] = h.z > 0.f ? w.z : 0.f; mk[4 * c + 3] = h.w > 0.f ? w.w : 0.f;
                    pr[c & 3] = fmaf(h.x, w.x, fmaf(h.y, w.y, fmaf(h.z, w.z, fmaf(h.w, w.w, pr[c & 3]))));   // eq. 3
                }
                const float pv = (pr[0] + pr[1]) + (pr[2] + pr[3]);
#pragma unroll
                for (uint32_t dd = 0; dd < C; ++dd) {          // one hop to every CTA of the cluster
                    const uint32_t d = (crank + dd) & (C - 1);
                    st_async_f32(mapa(ypp_a + (buf * (NSL * BT) + (crank * NTH + hb) * BT + frow) * 4, d), pv, mapa(yp_a + 8 * buf, d));
                }
            }
            // ---------------- eq. 5, eq. 7 ----------------
            mbar_wait(bar_yp + 8 * buf, ph);
            {
                const float* ypt = ypp + buf * (NSL * BT);
                float ypc[NSL];
#pragma unroll
                for (int c = 0; c < NSL; ++c) ypc[c] = ypt[c * BT + frow];
#pragma unroll
                for (int o = 1; o < NSL; o <<= 1)              // fixed pairwise tree over the partial slots
#pragma unroll
                    for (int c = 0; c + o < NSL; c += 2 * o) ypc[c] += ypc[c + o];
                const float d = frow < vt ? scale * (ypc[0] - ycur) : 0.f;
                if (hb == 0) Ds[frow] = d;
                if constexpr (BF16) {
                    float dz[32];
#pragma unroll
                    for (int u = 0; u < 32; ++u) dz[u] = d * mk[u];
#pragma unroll
                    for (int c = 0; c < 4; ++c)                // this row of dZ1 (64 units x 2 B = 128 bytes; S = 32: the upper half stays 0)
                        *reinterpret_cast<uint4*>(At + swz(frow, 4 * hb + c)) = pack_bf16x8(dz + 8 * c);
                } else {
                    // this row of dZ1 (32 units = 128 bytes): A operand of eq. 8, MN-major.  Rows r and r + 4 share a
                    // swizzle phase, so they store the two 16-byte halves of a 32-byte chunk in opposite order: the 8 rows
                    // of a quarter-warp then hit 8 different bank groups (no conflict) at the price of 4 selects per store
                    const bool flip = (frow >> 2) & 1;
#pragma unroll
                    for (int c = 0; c < 8; ++c) {
                        const int g = c >> 1, h0 = c & 1;      // logical chunk, half taken by the rows that do not flip
                        const float4 lo = make_float4(d * mk[8 * g], d * mk[8 * g + 1], d * mk[8 * g + 2], d * mk[8 * g + 3]);
                        const float4 hi = make_float4(d * mk[8 * g + 4], d * mk[8 * g + 5], d * mk[8 * g + 6], d * mk[8 * g + 7]);
                        const bool hsel = (h0 != 0) != flip;   // which half this thread stores now
                        *reinterpret_cast<float4*>(At + hb * (BT * 128) + swz32(frow, g, hsel ? 1 : 0)) = hsel ? hi : lo;
                    }
                }
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // At (generic writes) -> MMA
            __syncthreads();
            // ---------------- eq. 8 on the tensor cores: dW1^T += dZ1^T X ----------------
            if (warp == 0) {
                tc_fence_after();
                if (elect_one()) {
                    if constexpr (BF16) {
                        // both operands MN-major, 16 tile rows (2,048 bytes) per MMA; B = the BF16 copy of the tile (N = 32: the first
                        // 64 bytes of its 128-byte rows)
                        const uint64_t adesc = smem_desc_sw128_mn16(smem_u32(At)), bdesc = smem_desc_sw128_mn16(smem_u32(Xb));
#pragma unroll
                        for (int k = 0; k < BT / 16; ++k)
                            mma_f16(tmem_base + 64, adesc + 128 * k, bdesc + 128 * k, idesc8 | kIdescAMajorMN | kIdescBMajorMN, (j | k) != 0);
                    } else {
                        if constexpr (FOLD) {
                            // the chain of tiny MMAs costs per instruction (~30 cycles each), so the two row halves of the tile
                            // go through it side by side: A = [dZ1 rows k | dZ1 rows 128 + k] (M = 64: two 32-element column
                            // blocks 16 KB apart in At), B = [X rows k | X rows 128 + k] (N = 64, likewise in the tile).  The
                            // diagonal blocks of D (rows 0-31 x columns 0-31, rows 32-63 x columns 32-63) are the two halves
                            // of dW1^T, summed in the epilogue; the off-diagonal blocks are not read.
                            const uint64_t adesc = smem_desc_sw128_a32(smem_u32(At), 128 * 128);
                            const uint64_t bdesc = smem_desc_sw128_a32(smem_u32(Xs) + xst * kXBytes, 128 * 128);
#pragma unroll
                            for (int k = 0; k < BT / 16; ++k)
                                mma_tf32(tmem_base + 64, adesc + 64 * k, bdesc + 64 * k, idesc8f | kIdescAMajorMN | kIdescBMajorMN, (j | k) != 0);
                        } else {
                        // both operands MN-major: 8 tile rows (1,024 bytes) per MMA; A = the two 32-unit planes of dZ1
                        const uint64_t adesc = smem_desc_sw128_a32(smem_u32(At), BT * 128);
                        const uint64_t bdesc = smem_desc_sw128_a32(smem_u32(Xs) + xst * kXBytes, 1024);
#pragma unroll
                        for (int k = 0; k < BT / 8; ++k)
                            mma_tf32(tmem_base + 64, adesc + 64 * k, bdesc + 64 * k, idesc8 | kIdescAMajorMN | kIdescBMajorMN, (j | k) != 0);
                        }
                    }
                    tc_commit(bar_mma2);
                    if constexpr (!BF16) tc_commit(bar_empty + 8 * xst);   // the tensor core was the only reader of the X tile
                }
                __syncwarp();
            }
            // meanwhile eq. 6 on the CUDA cores: one unit per lane, 32 rows of the tile per warp
            {
                const int rbase = NTH == 1 ? warp * 32 : wq * 32;
                const unsigned char* Hh = Hs + hb * (BT * 128);
                float gp[4] = {0.f, 0.f, 0.f, 0.f};            // four independent chains hide the LDS latency
#pragma unroll
                for (int r = 0; r < 32; ++r) {
                    const int row = rbase + r;
                    gp[r & 3] = fmaf(*reinterpret_cast<const float*>(Hh + swz(row, lane >> 2) + (lane & 3) * 4), Ds[row], gp[r & 3]);
                }
                g2 += (gp[0] + gp[1]) + (gp[2] + gp[3]);
            }
            ycur = ynext;
            mbar_wait(bar_mma2, gt & 1u);                      // eq. 8 of this tile has read At and the tile
            tc_fence_after();
            __syncthreads();                                   // and every warp is done with Hs / Ds
        }

        // ---------------- end of batch: eq. 9 ----------------
        part2[warp * 32 + lane] = g2;
        if constexpr (FOLD) {
            // second diagonal block of the folded eq. 8: accumulator rows 32-63 (lanes 0-15 of warps 2, 3), columns 32-63;
            // handed to the owners of rows 0-31 through the (now idle) H buffer, 128-byte rows, chunks swizzled by lane
            if (warp == 2 || warp == 3) {
                uint32_t dh[32];
                tmem_ld32(tdw + 32, dh);
                tmem_ld_wait();
                tc_fence_before();
                if (lane < 16) {
#pragma unroll
                    for (int c = 0; c < 8; ++c)
                        *reinterpret_cast<uint4*>(Hs + ((warp - 2) * 16 + lane) * 128 + ((c ^ (lane & 7)) << 4)) =
                            make_uint4(dh[4 * c], dh[4 * c + 1], dh[4 * c + 2], dh[4 * c + 3]);
                }
            }
        }
        __syncthreads();
        if (warp < S / 16) {                                   // owners of the eq. 8 accumulator rows
            uint32_t dw[32];
            tmem_ld32(tdw, dw);
            tmem_ld_wait();
            tc_fence_before();
            if constexpr (FOLD) {
                if (wowner) {
#pragma unroll
                    for (int c = 0; c < 8; ++c) {
                        const float4 v = *reinterpret_cast<const float4*>(Hs + wu * 128 + ((c ^ (lane & 7)) << 4));
                        dw[4 * c] = __float_as_uint(__uint_as_float(dw[4 * c]) + v.x);
                        dw[4 * c + 1] = __float_as_uint(__uint_as_float(dw[4 * c + 1]) + v.y);
                        dw[4 * c + 2] = __float_as_uint(__uint_as_float(dw[4 * c + 2]) + v.z);
                        dw[4 * c + 3] = __float_as_uint(__uint_as_float(dw[4 * c + 3]) + v.w);
                    }
                }
            }
            if (wowner) {
#pragma unroll
                for (int i = 0; i < kIn; ++i) wrow[i] = fmaf(-p.lr, __uint_as_float(dw[i]), wrow[i]);   // W - lr*dW
                store_wop();
            }
        } else if (warp >= 4 && warp < 4 + S / 32) {           // meanwhile eq. 9 for W2 (one unit per lane)
            const int hbw = warp - 4;                          // S = 32: warp 4, all 8 row blocks; S = 64: warps 4, 5
            float sum = 0.f;
            if constexpr (NTH == 1) {
#pragma unroll
                for (int w = 0; w < kWarps; ++w) sum += part2[w * 32 + lane];
            } else {
#pragma unroll
                for (int q = 0; q < 4; ++q) sum += part2[(hbw * 4 + q) * 32 + lane];
            }
            W2s[hbw * 32 + lane] -= p.lr * sum;
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

// hidden 32..256: 32 units per CTA on hidden/32 CTAs; hidden 512 / 1024: 64 units per CTA on 8 / 16 CTAs
bool train_tc_supported(int hidden, bool bf16) {
    (void)bf16;
    return hidden == 32 || hidden == 64 || hidden == 128 || hidden == 256 || hidden == 512 || hidden == 1024;
}

namespace {

template <int C, int S, bool BF16>
cudaError_t launch_one(const float* X, int64_t n, const TcParams& p, cudaStream_t stream) {
    using P = TcPlan<C, S, BF16>;
    static_assert(P::BYTES <= 227 * 1024, "shared-memory plan exceeds the per-CTA limit");
    if (n > 0x7fffffffLL - P::BT) return cudaErrorInvalidValue;          // TMA coordinates are int32
    alignas(64) CUtensorMap tmap;
    if (!make_x_tensormap(&tmap, X, n, P::BT, /*atom32=*/!BF16)) return cudaErrorNotSupported;
    auto kern = k_train_tc<C, S, BF16>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P::BYTES);
    if (e != cudaSuccess) return e;
    if (C > 8) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e != cudaSuccess) return e;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(C);
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = P::BYTES;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = C;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, tmap, p);
}

template <bool BF16>
cudaError_t launch_width(const float* X, int64_t n, const TcParams& p, int hidden, cudaStream_t stream) {
    switch (hidden) {
        case 32: return launch_one<1, 32, BF16>(X, n, p, stream);
        case 64: return launch_one<2, 32, BF16>(X, n, p, stream);
        case 128: return launch_one<4, 32, BF16>(X, n, p, stream);
        case 256: return launch_one<8, 32, BF16>(X, n, p, stream);
        case 512: return launch_one<8, 64, BF16>(X, n, p, stream);
        case 1024: return launch_one<16, 64, BF16>(X, n, p, stream);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace

cudaError_t launch_train_tc(const float* X, const float* Y, int64_t n, int batch, float lr, int epochs,
                            float* W1, float* W2, const int32_t* order, int hidden, bool bf16,
                            unsigned long long* stats, cudaStream_t stream, int64_t* launches) {
    if (!train_tc_supported(hidden, bf16)) return cudaErrorInvalidValue;
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
    const cudaError_t err = bf16 ? launch_width<true>(X, n, p, hidden, stream) : launch_width<false>(X, n, p, hidden, stream);
    if (err == cudaSuccess) ++*launches;
    return err;
}

}  // namespace mlp
