// eval_tc.cu -- tensor-core variants of the eval pass (SURVEY.md 8(a) rows a-E / a-T, 8(f) NEXT-1):
//   L = (1/n) sum_r (ReLU(X_r W1) W2 - Y_r)^2          (eqs. 1-4)
// with eq. 1 on the 5th-generation tensor cores (tcgen05.mma, fp32 accumulate in TMEM).  Three operand
// modes, each a separately reported variant with its own tolerance:
//   TF32    kind::tf32: the fp32 operands are read straight from shared memory and truncated to TF32 by the
//           tensor core (loss within 1 % of the oracle; measured <= 4e-4);
//   BF16    kind::f16 with BF16 operands: four converter warps round the landed X tile to BF16 in place
//           (round to nearest even), half the tensor time per sample (loss within 1 %; measured <= 1e-4);
//   TF32X3  three TF32 products X W + (X - trunc X) W + X (W - trunc W): the converter warps write the
//           residual tile beside the landed one; fp32-faithful (loss within 1e-5).
// This is what makes the pass HBM-bound -- the exact-fp32 kernel is bound by the FP32 pipes at 128 FLOP/B.
//
// Persistent grid, one CTA per SM, warp-specialised:
//   warp 0      TMA producer: 128-row X tiles (16 KB) by cp.async.bulk.tensor with the 128-byte
//               swizzle the MMA wants, into a kStages-deep ring; in the BF16 / TF32X3 modes this warp
//               and warp 11 convert every landed tile (half a tile each, a lane owns two rows) before
//               the MMA may read it (more converter warps would cap the epilogue's registers at 128);
//   warp 1, 10  MMA issuers (even / odd tiles): per tile and column part four tcgen05.mma
//               (M=128, N=hidden/NH, K=8) into the TMEM accumulator of that tile parity
//               (2 x 256 columns = all of TMEM); tcgen05.commit releases the ring slot and
//               publishes the accumulator part.  One issuer per accumulator, so an epilogue set
//               never waits behind the other set's hand-back;
//   warps 2-9   epilogue, two sets of four warps (even / odd tiles, one TMEM accumulator each):
//               a thread owns one row, streams its hidden row out of TMEM (tcgen05.ld 32x32b),
//               applies eqs. 2-3 (ReLU + signed sum: |W2| is folded into the B operand, see
//               "setup"), eq. 4 in compensated fp32 per thread, fp64 from the warp level up.
//               Deterministic: fixed-order block and last-block reductions.
// W1 diag|W2| is transposed once per CTA into the K-major swizzled B operand ([hidden][32] floats).
// hidden > 256: 256-column slices of the same X tile alternate between the two accumulators.
#include <cuda.h>

#include "tc_common.cuh"

namespace mlp {
namespace {

constexpr int kTile = 128;           // rows per MMA (M)
constexpr int kStages = 6;           // X ring depth (6 x 16 KB)
constexpr int kEvalThreads = 352;    // producer + MMA (even tiles) + 8 epilogue warps + MMA (odd tiles)
constexpr int kEvalThreadsConv = 384; // + the second converter warp of the BF16 / TF32X3 modes
enum { kModeTf32 = 0, kModeBf16 = 1, kModeTf32x3 = 2 };
constexpr uint32_t kTileBytes = kTile * kIn * 4;

// Hidden widths above 256 (one MMA N-extent, half of TMEM) are processed as NS = H/256 column
// slices per tile: the X tile is read from HBM once, slice sl of a tile goes to accumulator
// (sl & 1), and the two epilogue sets combine their per-row partial sums through shared memory.
constexpr int eval_stages(int H, int mode) { return (H >= 1024 || mode == kModeTf32x3) ? 4 : kStages; }

template <int H, int MODE>
__global__ void __launch_bounds__(MODE == kModeTf32 ? kEvalThreads : kEvalThreadsConv, 1)
k_eval_tc(const __grid_constant__ CUtensorMap tmapX, const float* __restrict__ Y, long long n,
            const float* __restrict__ W1, const float* __restrict__ W2,
            double* __restrict__ partials, unsigned int* __restrict__ ticket,
            double* __restrict__ out) {
    static_assert(H % 32 == 0 && H >= 32 && H <= 1024 && (H <= 256 || H % 256 == 0), "hidden width");
    constexpr int HS = H < 256 ? H : 256;      // columns per slice (one MMA N-extent at most)
    constexpr int NS = H / HS;                 // slices per tile (1, 2 or 4)
    // Each 256-column TMEM accumulator is filled and drained in NH column parts, so the MMA of the
    // next item's first part overlaps the epilogue of this item's second part.
    constexpr int NH = HS >= 128 ? 2 : 1;
    constexpr int CP = HS / NH;                // columns (hidden units) per part
    constexpr int NST = eval_stages(H, MODE);  // X ring depth
    constexpr int NB = MODE == kModeTf32x3 ? 2 : 1;       // operand copies (value, residual)
    static_assert(MODE != kModeTf32x3 || H <= 256, "the three-product mode keeps two copies of both operands");
    constexpr int NG = H / 32;                 // 32-unit groups
    // 1024-byte alignment: swizzle atoms of both operands (checked below)
    extern __shared__ __align__(1024) unsigned char smem[];
    float* Bs = reinterpret_cast<float*>(smem);                            // [NB][H][128 B] swizzled rows (fp32 or bf16)
    unsigned char* Xring = smem + NB * H * kIn * 4;                        // [NB][NST][16 KB]
    uint64_t* bars = reinterpret_cast<uint64_t*>(Xring + NB * NST * kTileBytes);   // full, empty, tfull[2][NH], tempty[2][NH], conv
    double* wsum = reinterpret_cast<double*>(bars + 3 * NST + 16);         // [8]
    float* rowpart = reinterpret_cast<float*>(wsum + 8);                   // [2][128] partial rows of set 1
    int* wcnt = reinterpret_cast<int*>(rowpart + 2 * kTile);               // [32]
    int* npos_s = wcnt + 32;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(npos_s + 1);
    const uint32_t bar_full = smem_u32(bars), bar_empty = smem_u32(bars + NST),
                   bar_tfull = smem_u32(bars + 2 * NST), bar_tempty = smem_u32(bars + 2 * NST + 8),
                   bar_conv = smem_u32(bars + 2 * NST + 16);               // [NST] tile converted (BF16 / TF32X3)

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    constexpr int NW = (MODE == kModeTf32 ? kEvalThreads : kEvalThreadsConv) / 32;
    __shared__ int last_flag_s;
    int* last_flag = &last_flag_s;

    // ---- setup -------------------------------------------------------------------------------------
    // W2 is folded into the B operand: column j of Z' = X (W1 diag|W2|) is |w2_j| z_j, and
    //   w2_j ReLU(z_j) = sign(w2_j) ReLU(z'_j),
    // so the epilogue needs no multiply and no W2 operand (the W2 loads used to take as many
    // shared-memory cycles as the MMA operand reads).  Hidden units are permuted so that every
    // 32-column chunk has one sign, except chunk 0, which collects the remainder of both signs and
    // is summed with +-1 weights kept in registers.  Columns 24..31 of every chunk take ReLU as
    // (z + |z|) on the FMA pipe and carry a factor 1/2.
    if (tid == 0) {
        for (int s = 0; s < NST; ++s) {
            mbar_init(bar_full + 8 * s, 1); mbar_init(bar_empty + 8 * s, NS > 1 ? 2 : 1);
            mbar_init(bar_conv + 8 * s, 2);
        }
        for (int b = 0; b < 8; ++b) { mbar_init(bar_tfull + 8 * b, 1); mbar_init(bar_tempty + 8 * b, 4); }
        fence_mbar_init();
    }
    __syncthreads();
    const long long ntiles = (n + kTile - 1) / kTile;
    const long long my_tiles = blockIdx.x < ntiles ? (ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    const uint32_t nt = (uint32_t)my_tiles;
    // the first ring fill does not depend on the weights: start it before the operand set-up below
    if (warp == 0 && elect_one()) {
        for (uint32_t i = 0; i < nt && i < (uint32_t)NST; ++i) {
            const long long row0 = (blockIdx.x + (long long)i * gridDim.x) * kTile;
            mbar_arrive_expect_tx(bar_full + 8 * i, kTileBytes);        // OOB rows are zero-filled, still counted
            tma_load_2d(smem_u32(Xring) + i * kTileBytes, &tmapX, 0, (int)row0, bar_full + 8 * i);
        }
    }
    __syncwarp();
    // the warp's first group: its W1 column loads are issued together with the W2 loads of the sign count, so
    // the two global round trips (cold after a flush of L2) overlap
    float wcol[kIn];
    if (warp < NG) {
#pragma unroll
        for (int k = 0; k < kIn; ++k) wcol[k] = __ldg(W1 + (size_t)k * H + warp * 32 + lane);
    }
    for (int g = warp; g < NG; g += NW) {                      // a warp per group of 32 hidden units
        const unsigned bal = __ballot_sync(0xffffffffu, __ldg(W2 + g * 32 + lane) >= 0.f);
        if (lane == 0) wcnt[g] = __popc(bal);
    }
    __syncthreads();
    for (int g = warp; g < NG; g += NW) {
        const int j0 = g * 32 + lane;
        // lane stages column j0 of W1: 32 independent coalesced loads in flight at once
        if (g != warp) {
#pragma unroll
            for (int k = 0; k < kIn; ++k) wcol[k] = __ldg(W1 + (size_t)k * H + j0);
        }
        const float w2v = __ldg(W2 + j0);
        const unsigned bal = __ballot_sync(0xffffffffu, w2v >= 0.f);
        int before = __popc(bal & ((1u << lane) - 1u)), total = 0;
        for (int w = 0; w < NG; ++w) { const int c = wcnt[w]; total += c; if (w < g) before += c; }
        // chunk 0 takes the first r0 units with w2 >= 0 and the first 32 - r0 with w2 < 0, the
        // other (npos - r0, a multiple of 32) non-negative ones follow, then the negative ones
        const int r0 = (total & 31) ? (total & 31) : (total > 0 ? 32 : 0);
        const int a = before, b = j0 - before;                          // rank among its sign
        const int j = w2v >= 0.f ? (a < r0 ? a : 32 + (a - r0))
                                 : (b < 32 - r0 ? r0 + b : total + b);  // permuted column = B row
        const float sc = ((j & 31) >= 24 ? 0.5f : 1.0f) * fabsf(w2v);
        if (j0 == 0) *npos_s = total;
        unsigned char* brow = smem + (j >> 3) * 1024 + (j & 7) * 128;    // K-major row, 128B swizzle
#pragma unroll
        for (int k = 0; k < kIn; ++k) wcol[k] *= sc;
        if constexpr (MODE == kModeBf16) {                               // 32 bf16 = the first 64 logical bytes of the row
#pragma unroll
            for (int c = 0; c < kIn / 8; ++c)
                *reinterpret_cast<uint4*>(brow + ((c ^ (j & 7)) << 4)) =
                    make_uint4(bf16x2(wcol[8 * c], wcol[8 * c + 1]), bf16x2(wcol[8 * c + 2], wcol[8 * c + 3]),
                               bf16x2(wcol[8 * c + 4], wcol[8 * c + 5]), bf16x2(wcol[8 * c + 6], wcol[8 * c + 7]));
        } else {
#pragma unroll
            for (int c = 0; c < kIn / 4; ++c) {
                if constexpr (MODE == kModeTf32x3)                       // value operand already exact in TF32
                    *reinterpret_cast<float4*>(brow + ((c ^ (j & 7)) << 4)) =
                        make_float4(tf32_trunc(wcol[4 * c]), tf32_trunc(wcol[4 * c + 1]), tf32_trunc(wcol[4 * c + 2]), tf32_trunc(wcol[4 * c + 3]));
                else
                    *reinterpret_cast<float4*>(brow + ((c ^ (j & 7)) << 4)) =
                        make_float4(wcol[4 * c], wcol[4 * c + 1], wcol[4 * c + 2], wcol[4 * c + 3]);
                if constexpr (MODE == kModeTf32x3)                       // what the truncation drops (exact in fp32)
                    *reinterpret_cast<float4*>(brow + H * 128 + ((c ^ (j & 7)) << 4)) =
                        make_float4(tf32_residual(wcol[4 * c]), tf32_residual(wcol[4 * c + 1]),
                                    tf32_residual(wcol[4 * c + 2]), tf32_residual(wcol[4 * c + 3]));
            }
        }
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot))
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // generic B writes -> async proxy (MMA)
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    const int npos = *npos_s;
    if (smem_u32(smem) & 1023u) __trap();

    double sse = 0.0;
    // Work items: item w = i * NS + sl is slice sl of this CTA's i-th tile; it uses accumulator
    // (w & 1), MMA issuer (w & 1) and epilogue set (w & 1).  nt * NS < 2^31 by the host check.
    const uint32_t nitems = nt * NS;

    // BF16 / TF32X3: warp 0 (rows 0-63) and warp 11 (rows 64-127) convert every landed tile, a lane owns two rows of its half
    auto convert_half = [&](uint32_t i, int half) {
        const uint32_t st = i % NST;
        mbar_wait(bar_full + 8 * st, (i / NST) & 1u);
#pragma unroll
        for (int rr = 0; rr < 2; ++rr) {
            const int r = half * 64 + rr * 32 + lane;
            unsigned char* row = Xring + st * kTileBytes + r * 128;
            float4 v[8];
#pragma unroll
            for (int c = 0; c < 8; ++c) v[c] = *reinterpret_cast<const float4*>(row + ((c ^ (r & 7)) << 4));
            if constexpr (MODE == kModeBf16) {                          // in place: 32 bf16 in the first 64 logical bytes
#pragma unroll
                for (int c = 0; c < 4; ++c)
                    *reinterpret_cast<uint4*>(row + ((c ^ (r & 7)) << 4)) =
                        make_uint4(bf16x2(v[2 * c].x, v[2 * c].y), bf16x2(v[2 * c].z, v[2 * c].w),
                                   bf16x2(v[2 * c + 1].x, v[2 * c + 1].y), bf16x2(v[2 * c + 1].z, v[2 * c + 1].w));
            } else {                                                    // value exact in TF32 in place, residual beside it
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    *reinterpret_cast<float4*>(row + ((c ^ (r & 7)) << 4)) =
                        make_float4(tf32_trunc(v[c].x), tf32_trunc(v[c].y), tf32_trunc(v[c].z), tf32_trunc(v[c].w));
                    *reinterpret_cast<float4*>(row + NST * kTileBytes + ((c ^ (r & 7)) << 4)) =
                        make_float4(tf32_residual(v[c].x), tf32_residual(v[c].y), tf32_residual(v[c].z), tf32_residual(v[c].w));
                }
            }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");    // generic writes -> MMA (async proxy)
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_conv + 8 * st);
    };
    if (warp == 0) {
        // ===== TMA producer (whole warp runs the loop, one elected lane issues) =====
        auto refill = [&](uint32_t i) {                 // tile i goes into the slot tile i - NST has left
            const uint32_t st = i % NST;
            mbar_wait(bar_empty + 8 * st, ((i / NST) - 1u) & 1u);
            if (elect_one()) {
                const long long row0 = (blockIdx.x + (long long)i * gridDim.x) * kTile;
                mbar_arrive_expect_tx(bar_full + 8 * st, kTileBytes);   // OOB rows are zero-filled, still counted
                tma_load_2d(smem_u32(Xring) + st * kTileBytes, &tmapX, 0, (int)row0, bar_full + 8 * st);
            }
            __syncwarp();
        };
        if constexpr (MODE == kModeTf32) {
            for (uint32_t i = NST; i < nt; ++i) refill(i);   // tiles 0..NST-1 were issued before the set-up
        } else {
            // ... and converter: tile i is converted as soon as it has landed; the slot of tile i - 1 is refilled
            // afterwards (its MMA has had a whole conversion to finish), so the two duties never wait on each other
            for (uint32_t i = 0; i < nt; ++i) {
                convert_half(i, 0);
                if (i >= 1 && i - 1 + NST < nt) refill(i - 1 + NST);
            }
        }
    } else if (warp == 11) {
        if constexpr (MODE != kModeTf32)
            for (uint32_t i = 0; i < nt; ++i) convert_half(i, 1);
    } else if (warp == 1 || warp == 10) {
        // ===== MMA issuers: warp 1 feeds accumulator 0 (even items), warp 10 accumulator 1 (odd items), so
        // that neither epilogue set ever waits behind the other set's TMEM hand-back (whole warp runs
        // the loop, one elected lane issues) =====
        // instruction descriptor: D=f32, A=B=tf32, both K-major, N=CP, M=128
        constexpr uint32_t idesc = mma_idesc(MODE == kModeBf16 ? 1u : 2u, kTile, CP);
        const uint64_t bdesc = smem_desc_sw128(smem_u32(Bs));
        const uint64_t adesc0 = smem_desc_sw128(smem_u32(Xring));
        const uint32_t b = warp == 1 ? 0u : 1u;
        for (uint32_t w = b, kth = 0; w < nitems; w += 2, ++kth) {
            const uint32_t i = w / NS, sl = w % NS, st = i % NST;
            const uint32_t tph = (kth - 1u) & 1u;
            mbar_wait((MODE == kModeTf32 ? bar_full : bar_conv) + 8 * st, (i / NST) & 1u);
            const uint64_t adesc = adesc0 + (uint64_t)(st * (kTileBytes >> 4));
#pragma unroll
            for (int hf = 0; hf < NH; ++hf) {
                if (kth >= 1) mbar_wait(bar_tempty + 8 * (NH * b + hf), tph);
                tc_fence_after();
                if (elect_one()) {
                    const uint32_t dcol = tmem_base + b * 256 + hf * CP;
                    const uint64_t bd = bdesc + (uint64_t)((sl * HS + hf * CP) * 128 / 16);
                    if constexpr (MODE == kModeBf16) {
#pragma unroll
                        for (int k = 0; k < kIn / 16; ++k)  // K = 16 bf16 = 32 bytes per MMA: +2 in 16-byte units
                            mma_f16(dcol, adesc + 2 * k, bd + 2 * k, idesc, k > 0);
                    } else {
#pragma unroll
                        for (int k = 0; k < kIn / 8; ++k)   // K = 8 tf32 = 32 bytes per MMA: +2 in 16-byte units
                            mma_tf32(dcol, adesc + 2 * k, bd + 2 * k, idesc, k > 0);
                        if constexpr (MODE == kModeTf32x3) {
                            constexpr uint64_t xl = (uint64_t)(NST * kTileBytes >> 4), bl = (uint64_t)(H * 128 >> 4);
#pragma unroll
                            for (int k = 0; k < kIn / 8; ++k)   // + (X - trunc X) trunc W
                                mma_tf32(dcol, adesc + xl + 2 * k, bd + 2 * k, idesc, 1u);
#pragma unroll
                            for (int k = 0; k < kIn / 8; ++k)   // + trunc X (W - trunc W)
                                mma_tf32(dcol, adesc + 2 * k, bd + bl + 2 * k, idesc, 1u);
                        }
                    }
                    // ring slot free once the last slice this issuer takes from the tile has read it
                    if (hf == NH - 1 && sl + 2 >= NS) tc_commit(bar_empty + 8 * st);
                    tc_commit(bar_tfull + 8 * (NH * b + hf));           // accumulator part ready
                }
                __syncwarp();
            }
        }
    } else {
        // ===== epilogue: set e drains the items w with (w & 1) == e; warp quarter q owns TMEM lanes 32q.. =====
        const int e = (warp - 2) >> 2, q = warp & 3;
        float sse32 = 0.f, comp = 0.f;
        const int r0 = (npos & 31) ? (npos & 31) : (npos > 0 ? 32 : 0);   // non-negative units in chunk 0
        f32x2 sgn0[16];                                                  // +-1 weights of chunk 0
#pragma unroll
        for (int t = 0; t < 16; ++t) sgn0[t] = pack2(2 * t < r0 ? 1.f : -1.f, 2 * t + 1 < r0 ? 1.f : -1.f);
        float yp = 0.f, yv = 0.f;
        for (uint32_t w = e, kth = 0; w < nitems; w += 2, ++kth) {
            const uint32_t i = w / NS, sl = w % NS;
            const long long row = (blockIdx.x + (long long)i * gridDim.x) * kTile + q * 32 + lane;
            if (sl < 2) {                                       // first slice this set takes from the tile
                yp = 0.f;
                yv = ((NS == 1 || e == 0) && row < n) ? __ldg(Y + row) : 0.f;
            }
#pragma unroll
            for (int hf = 0; hf < NH; ++hf) {
                mbar_wait(bar_tfull + 8 * (NH * e + hf), kth & 1u);
                tc_fence_after();
                const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + e * 256 + hf * CP;
                uint32_t z[2][32];
                tmem_ld32(taddr, z[0]);
                tmem_ld_wait();
#pragma unroll
                for (int c = 0; c < CP / 32; ++c) {
                    if (c + 1 < CP / 32) tmem_ld32(taddr + (c + 1) * 32, z[(c + 1) & 1]);
                    const int cb = (int)sl * HS + hf * CP + c * 32;             // first (permuted) column
                    const float* zc = reinterpret_cast<const float*>(z[c & 1]);
                    // chunk 0 of the permuted order (columns 0..31) holds both signs
                    const bool mixed = hf == 0 && c == 0 && (NS == 1 || sl == 0);
                    f32x2 sc[4];
                    if (hf == 0 && c == 0 && mixed) {
#pragma unroll
                        for (int t = 0; t < 32; t += 2) {                       // signed sum
                            const float h0 = t < 24 ? fmaxf(zc[t], 0.f) : zc[t] + fabsf(zc[t]);
                            const float h1 = t < 24 ? fmaxf(zc[t + 1], 0.f) : zc[t + 1] + fabsf(zc[t + 1]);
                            const int a4 = (t >> 1) & 3;
                            if (t < 8) sc[a4] = fmul2(pack2(h0, h1), sgn0[t >> 1]);
                            else ffma2(sc[a4], pack2(h0, h1), sgn0[t >> 1]);
                        }
                    } else {
#pragma unroll
                        for (int t = 0; t < 32; t += 2) {                       // eq. 2 on two pipes
                            const float h0 = t < 24 ? fmaxf(zc[t], 0.f) : zc[t] + fabsf(zc[t]);
                            const float h1 = t < 24 ? fmaxf(zc[t + 1], 0.f) : zc[t + 1] + fabsf(zc[t + 1]);
                            const int a4 = (t >> 1) & 3;
                            sc[a4] = t < 8 ? pack2(h0, h1) : fadd2(sc[a4], pack2(h0, h1));
                        }
                    }
                    const float csum = hsum2(fadd2(fadd2(sc[0], sc[1]), fadd2(sc[2], sc[3])));
                    if (mixed) yp += csum;                                       // signs applied per column
                    else yp = fmaf(cb - 32 < npos - r0 ? 1.f : -1.f, csum, yp);  // eq. 3: sign of the chunk
                    if (c + 1 < CP / 32) tmem_ld_wait();
                    if (c + 2 == CP / 32 || CP == 32) {
                        // every column of this part is now in registers: hand it back to the MMA warp
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive(bar_tempty + 8 * (NH * e + hf));
                    }
                }
            }
            if (sl + 2 < NS) continue;                          // more slices of this tile for this set
            if constexpr (NS > 1) {
                // the two sets hold the two halves of the row sum: set 1 hands its half to set 0
                float* rp = rowpart + (i & 1u) * kTile + q * 32 + lane;
                if (e == 1) *rp = yp;
                asm volatile("bar.sync %0, 64;" ::"r"(1 + q) : "memory");
                if (e == 0) yp += *rp;
                if (e == 1) continue;
            }
            const float err = row < n ? yp - yv : 0.f;
            const float t = fmaf(err, err, -comp);                             // eq. 4, Kahan-compensated fp32
            const float su = sse32 + t;
            comp = (su - sse32) - t;
            sse32 = su;
        }
        sse = (double)sse32;
        for (int o = 16; o > 0; o >>= 1) sse += __shfl_down_sync(0xffffffffu, sse, o);
        if (lane == 0) wsum[warp - 2] = sse;
    }

    // ---- teardown: fixed-order block reduction, last block finishes, TMEM freed -------------------
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        __syncwarp();
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
    }
    if (tid == 0) {
        double tot = 0.0;
        for (int w = 0; w < 8; ++w) tot += wsum[w];
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

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

// The driver entry point is looked up through the runtime, so the library does not link libcuda.
EncodeTiledFn encode_tiled() {
    static EncodeTiledFn fn = []() -> EncodeTiledFn {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) != cudaSuccess ||
            qres != cudaDriverEntryPointSuccess)
            return nullptr;
        return reinterpret_cast<EncodeTiledFn>(p);
    }();
    return fn;
}

template <int H, int MODE>
cudaError_t launch_hm(const CUtensorMap& tmap, const float* Y, long long n, const float* W1, const float* W2,
                      double* partials, unsigned int* ticket, int grid, double* d_out, cudaStream_t stream) {
    auto kern = k_eval_tc<H, MODE>;
    constexpr int NB = MODE == kModeTf32x3 ? 2 : 1;
    constexpr int NST = eval_stages(H, MODE);
    const size_t smem = (size_t)NB * H * kIn * 4 + (size_t)NB * NST * kTileBytes + 8 * (3 * NST + 16) + 8 * 8 + 2 * kTile * 4 +
                        32 * 4 + 4 + 4 + 64;
    cudaError_t err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err != cudaSuccess) return err;
    kern<<<grid, MODE == kModeTf32 ? kEvalThreads : kEvalThreadsConv, smem, stream>>>(tmap, Y, n, W1, W2, partials, ticket, d_out);
    return cudaGetLastError();
}

template <int H>
cudaError_t launch_h(int mode, const CUtensorMap& tmap, const float* Y, long long n, const float* W1, const float* W2,
                     double* partials, unsigned int* ticket, int grid, double* d_out, cudaStream_t stream) {
    if (mode == kModeBf16) return launch_hm<H, kModeBf16>(tmap, Y, n, W1, W2, partials, ticket, grid, d_out, stream);
    if constexpr (H <= 256)
        if (mode == kModeTf32x3) return launch_hm<H, kModeTf32x3>(tmap, Y, n, W1, W2, partials, ticket, grid, d_out, stream);
    return launch_hm<H, kModeTf32>(tmap, Y, n, W1, W2, partials, ticket, grid, d_out, stream);
}

}  // namespace

bool make_x_tensormap(void* out_map, const float* X, int64_t n, int box_rows, bool atom32) {
    EncodeTiledFn enc = encode_tiled();
    if (!enc) return false;
    const cuuint64_t dims[2] = {(cuuint64_t)kIn, (cuuint64_t)n};
    const cuuint64_t strides[1] = {(cuuint64_t)kIn * 4};
    const cuuint32_t box[2] = {(cuuint32_t)kIn, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1, 1};
    return enc(static_cast<CUtensorMap*>(out_map), CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(X),
               dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               atom32 ? CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B : CU_TENSOR_MAP_SWIZZLE_128B,
               CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// variant numbers of include/mlp.h: 2 = MLP_VARIANT_TF32, 5 = MLP_VARIANT_BF16, 6 = MLP_VARIANT_TF32X3
bool eval_tc_supported(int hidden, int variant) {
    const bool width = hidden == 32 || hidden == 64 || hidden == 128 || hidden == 256 || hidden == 512 || hidden == 1024;
    if (variant == 2 || variant == 5) return width;
    if (variant == 6) return width && hidden <= 256;
    return false;
}

cudaError_t launch_eval_tc(const float* X, const float* Y, int64_t n, const float* W1, const float* W2,
                           int hidden, int variant, double* partials, unsigned int* ticket, int grid, double* d_out,
                           cudaStream_t stream, int64_t* launches) {
    if (!eval_tc_supported(hidden, variant)) return cudaErrorInvalidValue;
    if (n > 0x7fffffffLL - kTile) return cudaErrorInvalidValue;      // TMA coordinates are int32
    const int mode = variant == 5 ? kModeBf16 : variant == 6 ? kModeTf32x3 : kModeTf32;
    // X as a 2-D tensor [n rows][32 floats]; box = one 128-row tile; 128-byte swizzle = the layout
    // tcgen05.mma reads a K-major operand in (a row is exactly one 128-byte swizzle span).
    CUtensorMap tmap;
    if (!make_x_tensormap(&tmap, X, n, kTile)) return cudaErrorNotSupported;
    cudaError_t err;
    switch (hidden) {
        case 32: err = launch_h<32>(mode, tmap, Y, n, W1, W2, partials, ticket, grid, d_out, stream); break;
        case 64: err = launch_h<64>(mode, tmap, Y, n, W1, W2, partials, ticket, grid, d_out, stream); break;
        case 128: err = launch_h<128>(mode, tmap, Y, n, W1, W2, partials, ticket, grid, d_out, stream); break;
        case 256: err = launch_h<256>(mode, tmap, Y, n, W1, W2, partials, ticket, grid, d_out, stream); break;
        case 512: err = launch_h<512>(mode, tmap, Y, n, W1, W2, partials, ticket, grid, d_out, stream); break;
        case 1024: err = launch_h<1024>(mode, tmap, Y, n, W1, W2, partials, ticket, grid, d_out, stream); break;
        default: return cudaErrorInvalidValue;
    }
    if (err == cudaSuccess) ++*launches;
    return err;
}

}  // namespace mlp
