// train_fused.cu -- persistent fused training kernel.
//
// One thread-block cluster of C CTAs (one per SM) runs EVERY SGD step of mlp_train in a single
// launch (PAPER.md:108-112 loop; eqs. 1-9).  The hidden dimension is split over
// the cluster: CTA c owns S = hidden/C hidden units, i.e. W1[:, cS:(c+1)S] and W2[cS:(c+1)S],
// whose fp32 master copy stays in shared memory for the whole run.
//
// Mapping inside a CTA (8 warps):
//   * a lane owns FOUR hidden units (u_j = lu + j*LPS, LPS = S/4 lanes per row); a warp instruction
//     covers SPW = 32/LPS rows (sub-groups s).  Lane id = bit 0 of s, then lu, then the other bits of
//     s: with this order both broadcast load patterns (X rows, W1 reload) cost 2 shared-memory
//     wavefronts per LDS.128.  The X tile is stored as SPW blocks of BT/SPW rows, block s shifted by
//     16*s bytes, so the SPW rows read by one LDS.128 fall into distinct bank groups;
//   * forward (eqs. 1-3), K-split over lane pairs: lane lu and its partner lu ^ LPS/2 share their
//     eight units and each takes one half of the 32 inputs: 8 columns x 16 inputs of W1 live in 128
//     registers for the forward pass only, half an X row is read per lane (4 LDS.128 feed 64 FFMA2,
//     fma.rn.f32x2) and the halves of Z1 meet by one shuffle per unit.  The first rows are processed
//     chunk-major so the register reload of W1 overlaps their FMAs.  H = ReLU(Z1) of the warp's rows
//     stays in registers between forward and backward;
//   * per-row partial Ypred: transposing shuffle tree over the LPS lanes, then pushed to every CTA
//     of the cluster with st.async (DSMEM store that completes transaction bytes on the
//     destination's mbarrier: one hop, no flag), one fixed peer per lane, straight-line code (the
//     cluster size is a template parameter).  A store carries the totals of up to four consecutive
//     rows (st.async .v4 / .v2): a quarter of the remote stores and of the barrier updates of
//     per-row stores, which is what the exchange of a 16-CTA cluster was bound by.  The tile is
//     processed as NSPLIT row groups so that the exchange of one group is in flight while the
//     other group computes;
//   * backward (eqs. 5-8), K-split over the sub-groups: every CTA sums the C partials (fixed tree)
//     -> dZ2; the lane of sub-group s accumulates dW1 only for inputs [IPS*s, IPS*(s+1)) of its four
//     units (32 registers at SPW = 4) but over the rows of ALL sub-groups, whose dZ1 arrives by
//     shuffle: no reduction across sub-groups.  Per-warp partials go to shared memory; at the end of
//     the batch the 8 warps' partials are summed by a fixed pairwise tree (deterministic) and eq. 9
//     is applied to the shared-memory master copy.
// X tiles arrive by cp.async.bulk (TMA engine) into a 3-stage ring, one tile ahead; Y one tile
// ahead into a holder lane's register.  Measured: DESIGN.md 5.1, profiles/r02_ncu.md; the cost model
// behind the mapping (loads and shuffles add to the FMA time): profiles/r02_microbench.md.
#include "common.cuh"
#include "internal.h"

namespace mlp {
namespace {

constexpr int kWarps = 8;
constexpr int kThreads = kWarps * 32;
constexpr int kRing = 3;      // X ring stages (prefetch distance 1, slack 1)

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
    // host-precomputed bookkeeping (keeps 64-bit arithmetic and divisions out of the step loop)
    int nbi;            // batches per epoch
    int m_last;         // rows of the last batch of an epoch (== B when B divides n)
    float scale_full;   // 2 / B       (eq. 5)
    float scale_last;   // 2 / m_last
};

template <int S, int BT, int NSPLIT, int C>
__global__ void __launch_bounds__(kThreads, 1) k_train_fused(const TrainParams p) {
    constexpr int LPS = S / 4;            // lanes per sample row
    constexpr int SPW = 32 / LPS;         // sample rows per warp instruction (row sub-groups)
    constexpr int RB = BT / SPW;          // rows per X block (one block per sub-group)
    constexpr int ITER = RB / kWarps;     // rows per lane per tile
    constexpr int ITS = ITER / NSPLIT;    // rows per lane per exchange sub-tile
    constexpr int XBLK = RB * kIn + 4;    // floats per X block incl. the 16-byte stagger
    constexpr int XSTAGE = SPW * XBLK;    // floats per ring stage
    static_assert(LPS >= 4 && LPS <= 32 && RB % kWarps == 0 && ITER >= 1 && ITER % NSPLIT == 0, "cfg");
    static_assert(ITS >= 1 && ITS <= LPS, "transposing reduction needs ITS <= LPS");
    // Ypred partials [2][C][BTP]: the rows of sub-group sp are shifted by sp * PADR floats, so that the
    // SPW rows one LDS.32 of the backward pass touches (RB rows apart: the same bank when RB % 32 == 0)
    // fall into different banks.
    constexpr int PADR = (SPW > 1 && RB % 32 == 0) ? 32 / SPW : 0;
    constexpr int BTP = BT + SPW * PADR;
    static_assert(PADR == 0 || ITS <= PADR, "padding must cover the rows of one exchange sub-tile");

    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    // lane <-> (row sub-group s, unit lane lu): bit 0 of s is bit 0 of the lane id, lu the next
    // log2(LPS) bits, the other bits of s above.  With this interleaving both kinds of broadcast
    // load cost 2 shared-memory wavefronts per LDS.128 (measured): the X loads (one address per
    // sub-group) and the W1 register reload (one address per lu, shared by the SPW sub-groups; with
    // lu in the low bits it costs 4).
    constexpr int LLPS = LPS == 4 ? 2 : LPS == 8 ? 3 : LPS == 16 ? 4 : 5;
    constexpr int LSH = SPW > 1 ? 1 : 0;                                   // position of lu in the lane id
    const int lu = (lane >> LSH) & (LPS - 1);
    const int s = SPW > 1 ? (lane & 1) | ((lane >> (1 + LLPS)) << 1) : 0;
    auto lane_of = [](int sg, int l) -> int { return SPW > 1 ? (sg & 1) | (l << 1) | ((sg >> 1) << (1 + LLPS)) : l; };
    const uint32_t crank = cluster_ctarank();   // C = cluster size (template: exchange code is straight-line)
    const int H = p.H;

    float* Xs = reinterpret_cast<float*>(smem_raw);          // [kRing][XSTAGE]
    constexpr int XRING = (kRing * XSTAGE + 31) / 32 * 32;    // floats; keeps what follows 128-byte aligned
    float* ypp = Xs + XRING;                                  // [2][C][BTP]
    float* part = ypp + 2 * C * BTP;                           // [kWarps][S*32]  layout [q][u][4]
    float* part2 = part + kWarps * S * kIn;                   // [kWarps][S]
    float* W1s = part2 + kWarps * S;                          // [S*32]          layout [q][u][4]
    float* W2s = W1s + S * kIn;                               // [S]
    uint64_t* bars = reinterpret_cast<uint64_t*>(W2s + S);    // full[kRing], empty[kRing], yp[2][NSPLIT]
    const uint32_t bar_full = smem_u32(bars), bar_empty = smem_u32(bars + kRing),
                   bar_yp = smem_u32(bars + 2 * kRing);

    unsigned long long clk0 = 0, ns0 = 0;
    if (crank == 0 && tid == 0) { clk0 = clock64(); ns0 = globaltimer_ns(); }

    // ---- one-time setup: zero the X ring, load this CTA's weight slice, init barriers ----------
    for (int f = tid; f < kRing * XSTAGE; f += kThreads) Xs[f] = 0.f;
    for (int f = tid; f < S * kIn; f += kThreads) {
        const int q = f / (S * 4), rem = f % (S * 4), u = rem >> 2, i = q * 4 + (rem & 3);
        W1s[f] = p.W1[(size_t)i * H + crank * S + u];
    }
    if (tid < S) W2s[tid] = p.W2[crank * S + tid];
    if (tid == 0) {
        for (int b = 0; b < kRing; ++b) {
            mbar_init(bar_full + 8 * b, 1);
            mbar_init(bar_empty + 8 * b, kWarps);
        }
        for (int b = 0; b < 2 * NSPLIT; ++b) mbar_init(bar_yp + 8 * b, 1);
        fence_mbar_init();
    }
    // generic-proxy zero fill of Xs must be ordered before the async-proxy bulk copies
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();
    cluster_sync_all();        // every CTA's barriers exist before anyone pushes to them

    const long long total = p.total_steps;
    // batch of a step: the order table, else sequential; `seq` counts steps modulo nb without division
    int seq = 0;                                      // (step + 2) % nb for the look-ahead below
    unsigned long long bad_order = 0;     // batch_order entries outside [0, nb): clamped, counted, reported
    // The table entry of step k is loaded when step k-3 starts and only looked at (range check) when
    // step k-2 starts, so the global-load latency never sits on a step's critical path.
    auto checked = [&](int t, int sq) -> int {
        if (!p.order) return sq;
        if ((unsigned)t < (unsigned)p.nbi) return t;
        ++bad_order;
        return t < 0 ? 0 : p.nbi - 1;
    };
    auto raw_entry = [&](long long step) -> int { return (p.order && step < total) ? __ldg(p.order + step) : 0; };
    auto rows_of = [&](int t) -> int { return t == p.nbi - 1 ? p.m_last : p.B; };
    // producer (one thread): bring `rows` rows starting at global row g0 into ring stage nbuf
    auto issue_tile = [&](long long g0, int rows, unsigned nbuf) {
        const uint32_t bar = bar_full + 8 * nbuf;
        mbar_arrive_expect_tx(bar, rows * 128);
#pragma unroll
        for (int b = 0; b < SPW; ++b) {
            const int rb = min(RB, rows - b * RB);
            if (rb > 0)
                bulk_g2s(smem_u32(Xs + nbuf * XSTAGE + b * XBLK), p.X + (g0 + b * RB) * kIn,
                         rb * 128, bar);
        }
    };
    int t_cur = checked(raw_entry(0), 0);
    int t_next = total > 1 ? checked(raw_entry(1), 1 % p.nbi) : 0;
    int raw2 = raw_entry(2);                          // entry of step + 2, not yet checked
    seq = 2 % p.nbi;
    if (warp == 0) {
        if (elect_one()) {
            const long long r0 = (long long)t_cur * p.B;
            const int m = rows_of(t_cur);
            issue_tile(r0, min(BT, m), 0);
        }
        __syncwarp();
    }

    const int rowl = warp * ITER;                     // first row of this lane inside its block
    // Ypred exchange: every lane pushes to one fixed peer (staggered by rank)
    constexpr int RPI = 32 / C;                       // segments served per push iteration (C <= 32)
    const uint32_t pd = ((lane & (C - 1)) + crank) & (C - 1);
    const uint32_t rem_ypp = mapa(smem_u32(ypp), pd), rem_bar = mapa(bar_yp, pd);
    constexpr int VW = ITS >= 4 ? 4 : ITS;            // rows per remote store (st.async .v4 / .v2 / scalar)
    constexpr int NSEG = ITS * SPW / VW;              // VW-row segments of a warp's exchange sub-tile
    constexpr int NPUSH = (NSEG * C + 31) / 32;
    float* mypart = part + warp * (S * kIn);
    // Targets: lane l < ITER*SPW of a warp holds Y of the warp's row (l / ITER, l % ITER); it is
    // fetched one tile ahead (global-load latency hidden by a whole tile) and handed to the lane
    // that computes dZ2 by a shuffle.
    const bool yholder = lane < ITER * SPW;
    const int yrow = (lane / ITER) * RB + rowl + (lane % ITER);
    float ycur = 0.f;
    {
        const long long r0 = (long long)t_cur * p.B;
        const int m = rows_of(t_cur);
        if (yholder && yrow < min(BT, m)) ycur = __ldg(p.Y + r0 + yrow);
    }
    unsigned gt = 0;   // global tile counter
    for (long long step = 0; step < total; ++step) {
        const int t_nn = (step + 2 < total) ? checked(raw2, seq) : 0;
        raw2 = raw_entry(step + 3);
        seq = seq + 1 == p.nbi ? 0 : seq + 1;
        const long long r0 = (long long)t_cur * p.B;
        const int m = rows_of(t_cur);
        const int ntiles = (m + BT - 1) / BT;
        const float scale = t_cur == p.nbi - 1 ? p.scale_last : p.scale_full;   // eq. 5: 2 / m
        float g2[4] = {0.f, 0.f, 0.f, 0.f};                   // dW2 partials (eq. 6)

        for (int j = 0; j < ntiles; ++j, ++gt) {
            const unsigned buf = gt & 1u, ph = (gt >> 1) & 1u;       // Ypred exchange buffers
            const unsigned xst = gt % kRing, xph = (gt / kRing) & 1u;   // X ring stage
            const int vt = min(BT, m - j * BT);               // valid rows in this tile
            const float* Xl = Xs + xst * XSTAGE + s * XBLK + rowl * kIn;   // this lane's rows
            const float* ypt = ypp + buf * (C * BTP);
            const int row0 = s * RB + rowl;                   // tile row of this lane's first row

            // next tile (uniform): the rest of this batch, else the first tile of the next batch
            long long nr0 = 0; int nrows = 0;
            if (j + 1 < ntiles) { nr0 = r0 + (long long)(j + 1) * BT; nrows = min(BT, m - (j + 1) * BT); }
            else if (step + 1 < total) {
                nr0 = (long long)t_next * p.B;
                nrows = min(BT, rows_of(t_next));
            }
            // Producer duties of warp 0: arm this tile's exchange barriers (transaction bytes that
            // arrive before the expectation are simply counted against it) and prefetch the next X
            // tile.  The whole warp takes the branch and one elected lane issues, so the bulk copies
            // are plain UBLKCP instructions instead of per-lane loops.
            auto producer_duties = [&]() {
                if (warp == 0) {
                    if (elect_one()) {
#pragma unroll
                        for (int q = 0; q < NSPLIT; ++q)
                            mbar_arrive_expect_tx(bar_yp + 8 * (buf * NSPLIT + q), C * (BT / NSPLIT) * 4);
                        if (nrows > 0) {
                            // the stage of tile gt+1 was last read by tile gt-2: released long ago
                            const unsigned g1 = gt + 1, nbuf = g1 % kRing;
                            if (g1 >= kRing) mbar_wait(bar_empty + 8 * nbuf, ((g1 / kRing) - 1) & 1u);
                            issue_tile(nr0, nrows, nbuf);
                        }
                    }
                    __syncwarp();
                }
            };
            producer_duties();
            float ynext = 0.f;
            if (yholder && yrow < nrows) ynext = __ldg(p.Y + nr0 + yrow);

            float hreg[ITER][4];
            float w2r[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) w2r[u] = W2s[lu + u * LPS];
            {
                // ---------------- forward: eqs. 1-3 (W1 columns in registers) ----------------
                // K-split over lane pairs: of the LPS lanes of a row, lane lu and its partner lu ^ LPS/2
                // share EIGHT hidden units (their own four each) and each takes one half of the 32
                // inputs.  A lane thus keeps 8 columns x 16 inputs of W1 in registers (the same 128 as
                // four whole columns), reads only half of an X row (4 LDS.128 instead of 8 for the same
                // 64 FFMA2: every byte a load returns to the register file costs FMA issue time), and
                // the two halves of Z1 meet by one shuffle per unit: a lane sends its partial of the
                // partner's units and receives the partner's partial of its own (no select: register
                // set 0 is always "my units", set 1 always "the partner's").
                // The weight registers are reloaded every step; the first rows are processed
                // chunk-major (4 inputs at a time) with each weight chunk loaded just ahead of its
                // FFMA2s, so the reload overlaps the FMAs instead of preceding them.
                constexpr int HL = LPS / 2;                  // lanes per input half
                constexpr int RP = 1;                        // rows processed together (more only adds register pressure)
                const int kh = lu / HL;                      // this lane's inputs: 16 kh .. 16 kh + 15
                const int pxor = HL << LSH;                  // lane-id distance to the partner
                f32x2 w[2][4][8];                            // [mine / partner's units][unit][input pair]
                const float* Wh = W1s + (4 * kh * S) * 4;
                auto load_w_chunk = [&](int c) {             // inputs 16 kh + 4c .. + 3 of the eight columns
#pragma unroll
                    for (int rel = 0; rel < 2; ++rel)
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            const int unit = (rel ? lu ^ HL : lu) + u * LPS;
                            const ulonglong2 a = *reinterpret_cast<const ulonglong2*>(Wh + (c * S + unit) * 4);
                            w[rel][u][2 * c] = a.x; w[rel][u][2 * c + 1] = a.y;
                        }
                };
                // one-row tiles (batches <= 32 rows) are latency-bound: the first weight chunk is requested before
                // the X tile is awaited (-3.5 % per step at B = 32; with more rows per lane it is a wash or a loss)
                if constexpr (ITER == 1) load_w_chunk(0);
                mbar_wait(bar_full + 8 * xst, xph);
                const float* Xh = Xl + 16 * kh;              // this lane's half of its rows
                if constexpr (ITER > 1) load_w_chunk(0);
#pragma unroll
                for (int q = 0; q < NSPLIT; ++q) {
                    float pv[ITS];
#pragma unroll
                    for (int k0 = 0; k0 < ITS; k0 += RP) {
                        f32x2 a[RP][2][4];
#pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            if (q == 0 && k0 == 0) {
                                if (c + 1 < 4) load_w_chunk(c + 1);
                                asm volatile("" ::: "memory");   // keep the later chunks' loads behind these FMAs
                            }
#pragma unroll
                            for (int r = 0; r < RP; ++r) {
                                const ulonglong2 xv = reinterpret_cast<const ulonglong2*>(Xh + (q * ITS + k0 + r) * kIn)[c];
#pragma unroll
                                for (int rel = 0; rel < 2; ++rel)
#pragma unroll
                                    for (int u = 0; u < 4; ++u) {
                                        if (c == 0) a[r][rel][u] = fmul2(xv.x, w[rel][u][0]);        // eq. 1
                                        else ffma2(a[r][rel][u], xv.x, w[rel][u][2 * c]);
                                        ffma2(a[r][rel][u], xv.y, w[rel][u][2 * c + 1]);
                                    }
                            }
                        }
#pragma unroll
                        for (int r = 0; r < RP; ++r) {
                            const int it = q * ITS + k0 + r;
#pragma unroll
                            for (int u = 0; u < 4; ++u) {
                                const float z = hsum2(a[r][0][u]) + __shfl_xor_sync(0xffffffffu, hsum2(a[r][1][u]), pxor);
                                hreg[it][u] = fmaxf(z, 0.f);                                         // eq. 2
                            }
                            pv[k0 + r] = fmaf(hreg[it][1], w2r[1], hreg[it][0] * w2r[0]) +           // eq. 3
                                         fmaf(hreg[it][3], w2r[3], hreg[it][2] * w2r[2]);
                        }
                    }
                    GroupReduce<ITS, LPS, 1, LSH>::run(pv, lu);
                    // push: lane l serves ONE destination CTA (pd) and the segments l/C, l/C + 32/C, ... of the
                    // warp's NSEG segments (VW consecutive rows of one sub-group), whose totals it fetches from
                    // their holder lanes by shuffle and sends as one 4*VW-byte store
#pragma unroll
                    for (int i = 0; i < NPUSH; ++i) {
                        const int r = lane / C + i * RPI;          // segment: VW consecutive rows of sub-group sp
                        const int sp = r / (ITS / VW), k0 = (r % (ITS / VW)) * VW;
                        float v[VW];
#pragma unroll
                        for (int k = 0; k < VW; ++k) v[k] = __shfl_sync(0xffffffffu, pv[0], lane_of(sp, k0 + k) & 31);
                        if (r < NSEG) {
                            const int row = sp * RB + rowl + q * ITS + k0;
                            const uint32_t dst = rem_ypp + (buf * (C * BTP) + crank * BTP + row + sp * PADR) * 4;
                            const uint32_t rb = rem_bar + 8 * (buf * NSPLIT + q);
                            if constexpr (VW == 4) st_async_v4(dst, v[0], v[1], v[2], v[3], rb);
                            else if constexpr (VW == 2) st_async_v2(dst, v[0], v[1], rb);
                            else st_async_f32(dst, v[0], rb);
                        }
                    }
                }
            }

            // ---------------- backward: eqs. 5-8 ----------------
            // K-split: the lane of sub-group s accumulates dW1 only for the IPS inputs
            // [IPS*s, IPS*(s+1)) of its four units, but over the rows of ALL sub-groups, so no
            // reduction across sub-groups is needed afterwards.  dZ1 of the other sub-groups'
            // rows arrives by shuffle; acc[u][kk] <-> inputs IPS*s + 2kk, +1.  (Rebuilding dZ1 locally
            // from one dZ2 shuffle per row and the owner lane's 32 ReLU' bits saves 70 % of the
            // shuffles but costs more issue slots than it frees: measured slower at C = 8.)
            constexpr int IPS = kIn / SPW;            // inputs per sub-group
            f32x2 acc[4][IPS / 2];
            const float* Xk = Xs + xst * XSTAGE + rowl * kIn + IPS * s;
#pragma unroll
            for (int q = 0; q < NSPLIT; ++q) {
                // The partials were written by st.async, whose completion is the barrier's
                // transaction count: the default (CTA-scope acquire) wait orders them; a
                // cluster-scope acquire would make ptxas emit CCTL.IVALL (L1 invalidate), which
                // stalls on every global load in flight.
                mbar_wait(bar_yp + 8 * (buf * NSPLIT + q), ph);
                float dzv;
                {
                    const int kk = lu & (ITS - 1);
                    const int row = row0 + q * ITS + kk;
                    const float yv = __shfl_sync(0xffffffffu, ycur, s * ITER + q * ITS + kk);
                    float ypc[C];
#pragma unroll
                    for (int c = 0; c < C; ++c) ypc[c] = ypt[c * BTP + row + s * PADR];
#pragma unroll
                    for (int o = 1; o < C; o <<= 1)                 // fixed pairwise tree over ranks
#pragma unroll
                        for (int c = 0; c + o < C; c += 2 * o) ypc[c] += ypc[c + o];
                    const float yp = ypc[0];
                    dzv = row < vt ? scale * (yp - yv) : 0.f;                 // eq. 5
                }
#pragma unroll
                for (int k = 0; k < ITS; ++k) {
                    const int it = q * ITS + k;
                    const float d = __shfl_sync(0xffffffffu, dzv, lane_of(s, k));
                    float e[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const float h = hreg[it][u];
                        g2[u] = fmaf(h, d, g2[u]);                             // eq. 6
                        e[u] = h > 0.f ? d * w2r[u] : 0.f;                     // eq. 7 (old W2)
                    }
#pragma unroll
                    for (int t = 0; t < SPW; ++t) {            // row of sub-group s ^ t
                        f32x2 dd[4];
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            const float eo = t == 0 ? e[u] : __shfl_xor_sync(0xffffffffu, e[u], lane_of(t, 0));
                            dd[u] = pack2(eo, eo);
                        }
                        const ulonglong2* xrow =
                            reinterpret_cast<const ulonglong2*>(Xk + (s ^ t) * XBLK + it * kIn);
#pragma unroll
                        for (int x = 0; x < IPS / 4; ++x) {                    // eq. 8
                            const ulonglong2 xv = xrow[x];
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
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_empty + 8 * xst);   // this warp is done with the X tile
            ycur = ynext;

            // lane (s, lu) owns the 4-input chunks q = (IPS/4)*s + x of its four units
            if (j == 0) {
#pragma unroll
                for (int u = 0; u < 4; ++u)
#pragma unroll
                    for (int x = 0; x < IPS / 4; ++x)
                        *reinterpret_cast<ulonglong2*>(mypart + (((IPS / 4) * s + x) * S + lu + u * LPS) * 4) =
                            make_ulonglong2(acc[u][2 * x], acc[u][2 * x + 1]);
            } else {                                           // later tiles of a large batch: accumulate
#pragma unroll
                for (int u = 0; u < 4; ++u)
#pragma unroll
                    for (int x = 0; x < IPS / 4; ++x) {
                        ulonglong2* dst =
                            reinterpret_cast<ulonglong2*>(mypart + (((IPS / 4) * s + x) * S + lu + u * LPS) * 4);
                        const ulonglong2 old = *dst;
                        *dst = make_ulonglong2(fadd2(acc[u][2 * x], old.x), fadd2(acc[u][2 * x + 1], old.y));
                    }
            }
        }

        // ---------------- end of batch: reduce partial gradients, eq. 9 ----------------
#pragma unroll
        for (int sb = 1; sb < SPW; sb <<= 1)                   // across the sub-groups (bits of s)
#pragma unroll
            for (int u = 0; u < 4; ++u) g2[u] += __shfl_xor_sync(0xffffffffu, g2[u], lane_of(sb, 0));
        if (s == 0) {
#pragma unroll
            for (int u = 0; u < 4; ++u) part2[warp * S + lu + u * LPS] = g2[u];
        }
        __syncthreads();
        {
            constexpr int NF = S * 8;                          // float4 slots of this CTA's dW1
            const f32x2 nlr2 = pack2(-p.lr, -p.lr);
#pragma unroll
            for (int r = 0; r < (NF + kThreads - 1) / kThreads; ++r) {
                const int f = tid + r * kThreads;
                if (NF % kThreads == 0 || f < NF) {
                    ulonglong2 v[kWarps];
#pragma unroll
                    for (int w = 0; w < kWarps; ++w)
                        v[w] = reinterpret_cast<const ulonglong2*>(part)[w * NF + f];
#pragma unroll
                    for (int o = 1; o < kWarps; o <<= 1)        // fixed pairwise tree over warps
#pragma unroll
                        for (int w = 0; w + o < kWarps; w += 2 * o) {
                            v[w].x = fadd2(v[w].x, v[w + o].x);
                            v[w].y = fadd2(v[w].y, v[w + o].y);
                        }
                    ulonglong2 wv = reinterpret_cast<ulonglong2*>(W1s)[f];
                    ffma2(wv.x, v[0].x, nlr2);                                 // eq. 9: W - lr*dW
                    ffma2(wv.y, v[0].y, nlr2);
                    reinterpret_cast<ulonglong2*>(W1s)[f] = wv;
                }
            }
        }
        if (tid < S) {
            float sum = part2[tid];
#pragma unroll
            for (int w = 1; w < kWarps; ++w) sum += part2[w * S + tid];
            W2s[tid] -= p.lr * sum;                                            // eq. 9
        }
        __syncthreads();
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
        p.stats[4] = bad_order;
    }
    cluster_sync_all();        // no CTA exits while peers may still push into its shared memory
}

template <int S, int BT, int C>
cudaError_t launch_cfg(const TrainParams& p, cudaStream_t stream) {
    constexpr int SPW = 32 / (S / 4);
    constexpr int ITER = BT / SPW / kWarps;
    constexpr int NSPLIT = ITER >= 2 ? 2 : 1;
    auto kern = k_train_fused<S, BT, NSPLIT, C>;
    constexpr int RB = BT / SPW;
    constexpr int BTP = BT + ((SPW > 1 && RB % 32 == 0) ? 32 : 0);      // padded Ypred exchange rows (see the kernel)
    const size_t smem = sizeof(float) * ((kRing * (BT * kIn + SPW * 4) + 31) / 32 * 32 + 2 * C * BTP +
                                         kWarps * S * kIn + kWarps * S + S * kIn + S) +
                        8 * (2 * kRing + 2 * NSPLIT);
    cudaError_t err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err != cudaSuccess) return err;
    if (C > 8) {
        err = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (err != cudaSuccess) return err;
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
    return cudaLaunchKernelEx(&cfg, kern, p);
}

// Tile height: the smallest instantiated height >= batch, else the largest (64*SPW rows, at most
// 256, keep H = ReLU(Z1) of a tile in 32 registers per lane).
template <int S, int C>
cudaError_t launch_sc(const TrainParams& p, cudaStream_t stream) {
    const int B = p.B;
    if constexpr (S == 16) {
        if (B > 64) return launch_cfg<16, 256, C>(p, stream);
        return launch_cfg<16, 64, C>(p, stream);
    } else if constexpr (S == 32) {
        if (B > 128) return launch_cfg<32, 256, C>(p, stream);
        if (B > 32) return launch_cfg<32, 128, C>(p, stream);
        return launch_cfg<32, 32, C>(p, stream);
    } else if constexpr (S == 64) {
        if (B > 32) return launch_cfg<64, 128, C>(p, stream);
        return launch_cfg<64, 32, C>(p, stream);
    } else {
        if (B > 32) return launch_cfg<128, 64, C>(p, stream);
        return launch_cfg<128, 32, C>(p, stream);
    }
}

// hidden = S * C must be one of 32..1024 (include/mlp.h): only those pairs are instantiated
template <int S>
cudaError_t launch_s(const TrainParams& p, int cluster, cudaStream_t stream) {
    switch (cluster) {
        case 1: if constexpr (S >= 32) return launch_sc<S, 1>(p, stream); break;
        case 2: return launch_sc<S, 2>(p, stream);
        case 4: return launch_sc<S, 4>(p, stream);
        case 8: return launch_sc<S, 8>(p, stream);
        case 16: if constexpr (S <= 64) return launch_sc<S, 16>(p, stream); break;
        default: break;
    }
    return cudaErrorInvalidValue;
}

}  // namespace

bool fused_supported(int hidden, int cluster) {
    if (cluster != 1 && cluster != 2 && cluster != 4 && cluster != 8 && cluster != 16) return false;
    if (hidden % cluster) return false;
    const int S = hidden / cluster;
    if (S == 16) return cluster >= 2;
    if (S == 128) return cluster <= 8;
    return S == 32 || S == 64;
}

int fused_default_cluster(int hidden, int batch) {
    (void)batch;
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
    p.nbi = (int)p.nb;
    p.m_last = (int)(n - (p.nb - 1) * batch);
    p.scale_full = 2.0f / (float)batch;
    p.scale_last = 2.0f / (float)p.m_last;
    p.W1 = W1; p.W2 = W2; p.order = order; p.H = hidden; p.stats = stats;
    if (p.total_steps == 0) return cudaSuccess;
    cudaError_t err;
    switch (hidden / cluster) {
        case 16: err = launch_s<16>(p, cluster, stream); break;
        case 32: err = launch_s<32>(p, cluster, stream); break;
        case 64: err = launch_s<64>(p, cluster, stream); break;
        case 128: err = launch_s<128>(p, cluster, stream); break;
        default: return cudaErrorInvalidValue;
    }
    if (err == cudaSuccess) ++*launches;
    return err;
}

}  // namespace mlp
