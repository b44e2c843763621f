/*
 * mlp_oracle.c -- CPU ORACLE for the mini-batch SGD step of the 32-256-1 ReLU/MSE MLP.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  The product
 * (paper_2606_30497_b200/, include/mlp.h) never does; it shares no code, header, helper
 * or constant table with this file.
 *
 * What it is: a plain, slow, obviously-correct restatement of PAPER.md eqs. 1-9
 * (restated as eqs. 11-19 at PAPER.md:123-154), followed step by step in
 * the paper's order.  Every sum is carried in fp64 in ascending index order; weights are
 * fp32 between steps (one rounding per weight per step, eq. 9).  Readings of the garbled
 * or silent passages are those of SURVEY.md 8(c) and are listed in DESIGN.md:
 *   - eq. 4 / eq. 14 (garbled): L = (1/n) sum_i (Ypred_i - Y_i)^2; eq. 5's 2/n is its derivative.
 *   - n in eq. 5 is the number of rows of the CURRENT mini-batch (m for a short tail batch).
 *   - ReLU'(x) = 1 if x > 0, otherwise 0: strict >, gradient 0 at 0.
 *   - eq. 7 uses W2 BEFORE this step's update (eqs. 6-8 precede eq. 9).
 *   - batches are contiguous row ranges [t*B, min(n,(t+1)*B)); `order` permutes batch indices.
 *   - lr is the fp32 value widened to double (not the double literal 0.002).
 *
 * Pins (tests/test_oracle_pins.py): P0 loop extents = PAPER.md:203-210 MAC counts;
 * P1/P2 hand-worked 2-sample/4-hidden example and the tie at zero (tests/golden/);
 * P3 finite differences; P4 lr=0; P5 descent identity; P6 linear closed form; P7 dead
 * network; P8 eval closed forms; P9 batch=n; P10 permutation invariance; P11 resume;
 * P12 torch-fp64 autograd; P13 brute force; P14 survey-time end-to-end losses.
 * Unpinned: parity with the AUTHORS' implementation (no code, no printed numeric result
 * other than timings exists) -- see DESIGN.md.
 *
 * OpenMP is used only where each thread owns whole output elements and sums them
 * sequentially in ascending index order, so results do not depend on the thread count.
 * Build: gcc -O2 -fno-fast-math -ffp-contract=off -fopenmp -shared -fPIC (oracle/build.py).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* MAC counters for pin P0, one per product: eq.1, eq.3, eq.6, eq.7, eq.8. */
enum { MAC_EQ1 = 0, MAC_EQ3 = 1, MAC_EQ6 = 2, MAC_EQ7 = 3, MAC_EQ8 = 4, MAC_N = 5 };

/*
 * One batch of m rows: forward (eqs. 1-3), loss (eq. 4), gradients (eqs. 5-8).
 * Xb [m x I] fp32 row-major, Yb [m] fp32, W1 [I x H] and W2 [H] in double (the caller
 * widens its fp32 weights exactly).  Outputs g1 [I x H], g2 [H], *loss (any may be NULL).
 * macs: NULL, or MAC_N counters incremented once per multiply-add (then runs serially).
 */
static void batch_grads(const float *Xb, const float *Yb, int m, int I, int H,
                        const double *W1, const double *W2,
                        double *g1, double *g2, double *loss, uint64_t *macs)
{
    double *z  = (double *)malloc(sizeof(double) * (size_t)m * H);   /* Z1, eq. 1 */
    double *h  = (double *)malloc(sizeof(double) * (size_t)m * H);   /* H,  eq. 2 */
    double *yp = (double *)malloc(sizeof(double) * (size_t)m);       /* Ypred, eq. 3 */
    double *d2 = (double *)malloc(sizeof(double) * (size_t)m);       /* dZ2, eq. 5 */
    double *d1 = (double *)malloc(sizeof(double) * (size_t)m * H);   /* dZ1, eq. 7 */
    const int serial = macs != NULL;

    /* eq. 1: Z1 = X W1 ;  eq. 2: H = ReLU(Z1) ;  eq. 3: Ypred = H W2 */
    #pragma omp parallel for schedule(static) if (!serial)
    for (int b = 0; b < m; ++b) {
        for (int j = 0; j < H; ++j) {
            double s = 0.0;
            for (int i = 0; i < I; ++i) {
                s += (double)Xb[(size_t)b * I + i] * W1[(size_t)i * H + j];
                if (serial) macs[MAC_EQ1]++;
            }
            z[(size_t)b * H + j] = s;
            h[(size_t)b * H + j] = s > 0.0 ? s : 0.0;
        }
        double y = 0.0;
        for (int j = 0; j < H; ++j) {
            y += h[(size_t)b * H + j] * W2[j];
            if (serial) macs[MAC_EQ3]++;
        }
        yp[b] = y;
    }

    /* eq. 4: L = (1/m) sum_b (Ypred_b - Y_b)^2 ;  eq. 5: dZ2 = (2/m)(Ypred - Y) */
    double sse = 0.0;
    for (int b = 0; b < m; ++b) {
        double e = yp[b] - (double)Yb[b];
        sse += e * e;
        d2[b] = (2.0 / (double)m) * e;
    }
    if (loss) *loss = sse / (double)m;

    if (g1 || g2) {
        /* eq. 6: dW2 = H^T dZ2 */
        if (g2) {
            #pragma omp parallel for schedule(static) if (!serial)
            for (int j = 0; j < H; ++j) {
                double s = 0.0;
                for (int b = 0; b < m; ++b) {
                    s += h[(size_t)b * H + j] * d2[b];
                    if (serial) macs[MAC_EQ6]++;
                }
                g2[j] = s;
            }
        }
        /* eq. 7: dZ1 = (dZ2 W2^T) (.) ReLU'(Z1), ReLU'(x) = 1 if x > 0 else 0; W2 is the
           pre-update W2 (this function never modifies it). */
        #pragma omp parallel for schedule(static) if (!serial)
        for (int b = 0; b < m; ++b) {
            for (int j = 0; j < H; ++j) {
                double t = d2[b] * W2[j];
                if (serial) macs[MAC_EQ7]++;
                d1[(size_t)b * H + j] = z[(size_t)b * H + j] > 0.0 ? t : 0.0;
            }
        }
        /* eq. 8: dW1 = X^T dZ1 */
        if (g1) {
            #pragma omp parallel for schedule(static) if (!serial)
            for (int j = 0; j < H; ++j) {
                for (int i = 0; i < I; ++i) {
                    double s = 0.0;
                    for (int b = 0; b < m; ++b) {
                        s += (double)Xb[(size_t)b * I + i] * d1[(size_t)b * H + j];
                        if (serial) macs[MAC_EQ8]++;
                    }
                    g1[(size_t)i * H + j] = s;
                }
            }
        }
    }
    free(z); free(h); free(yp); free(d2); free(d1);
}

/* Gradients and loss of one batch at double-precision weights (finite-difference pins). */
void oracle_grads_f64(const float *Xb, const float *Yb, int m, int I, int H,
                      const double *W1, const double *W2,
                      double *g1, double *g2, double *loss, uint64_t *macs)
{
    batch_grads(Xb, Yb, m, I, H, W1, W2, g1, g2, loss, macs);
}

/* Same at fp32 weights (widened exactly). */
void oracle_grads(const float *Xb, const float *Yb, int m, int I, int H,
                  const float *W1, const float *W2,
                  double *g1, double *g2, double *loss, uint64_t *macs)
{
    double *w1 = (double *)malloc(sizeof(double) * (size_t)I * H);
    double *w2 = (double *)malloc(sizeof(double) * (size_t)H);
    for (size_t k = 0; k < (size_t)I * H; ++k) w1[k] = (double)W1[k];
    for (int j = 0; j < H; ++j) w2[j] = (double)W2[j];
    batch_grads(Xb, Yb, m, I, H, w1, w2, g1, g2, loss, macs);
    free(w1); free(w2);
}

/*
 * Mini-batch SGD (PAPER.md:108-112 loop; eq. 9 update) over `epochs` x nb batches.
 * X [n x I], Y [n] fp32; W1 [I x H], W2 [H] fp32, updated in place.
 * order: NULL (sequential) or int32 [epochs x nb] batch indices.
 * state_fp64 != 0 keeps the weights in double ACROSS steps (drift report only, not a gate).
 * macs: NULL or MAC_N counters.  Returns the number of SGD steps taken, or -1 on bad args.
 */
int64_t oracle_train(const float *X, const float *Y, int64_t n, int I, int H, int B,
                     float lr, int epochs, float *W1, float *W2,
                     const int32_t *order, int state_fp64, uint64_t *macs)
{
    if (n < 1 || I < 1 || H < 1 || B < 1 || epochs < 0) return -1;
    const double a = (double)lr;                       /* widen the fp32 learning rate */
    const int64_t nb = (n + B - 1) / B;
    const size_t n1 = (size_t)I * H;
    double *w1 = (double *)malloc(sizeof(double) * n1);
    double *w2 = (double *)malloc(sizeof(double) * (size_t)H);
    double *g1 = (double *)malloc(sizeof(double) * n1);
    double *g2 = (double *)malloc(sizeof(double) * (size_t)H);
    for (size_t k = 0; k < n1; ++k) w1[k] = (double)W1[k];
    for (int j = 0; j < H; ++j) w2[j] = (double)W2[j];
    int64_t steps = 0;
    for (int e = 0; e < epochs; ++e) {
        for (int64_t k = 0; k < nb; ++k) {
            const int64_t t  = order ? (int64_t)order[(int64_t)e * nb + k] : k;
            const int64_t r0 = t * B;
            const int m = (int)((n - r0) < B ? (n - r0) : B);   /* rows in this batch */
            batch_grads(X + r0 * I, Y + r0, m, I, H, w1, w2, g1, g2, NULL, macs);
            /* eq. 9: W <- W - alpha dW, both matrices, after both gradients */
            for (size_t q = 0; q < n1; ++q) {
                double v = w1[q] - a * g1[q];
                w1[q] = state_fp64 ? v : (double)(float)v;      /* fp32 state: one rounding */
            }
            for (int j = 0; j < H; ++j) {
                double v = w2[j] - a * g2[j];
                w2[j] = state_fp64 ? v : (double)(float)v;
            }
            ++steps;
        }
    }
    for (size_t k = 0; k < n1; ++k) W1[k] = (float)w1[k];
    for (int j = 0; j < H; ++j) W2[j] = (float)w2[j];
    free(w1); free(w2); free(g1); free(g2);
    return steps;
}

/* eq. 4 over a whole dataset: L = (1/n) sum_r (relu(X_r W1) W2 - Y_r)^2, fp64, ascending r.
 * Each thread computes whole rows' squared errors into se[r]; the final sum is serial. */
double oracle_eval_loss(const float *X, const float *Y, int64_t n, int I, int H,
                        const float *W1, const float *W2)
{
    if (n < 1) return NAN;
    double *se = (double *)malloc(sizeof(double) * (size_t)n);
    #pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < n; ++r) {
        double y = 0.0;
        for (int j = 0; j < H; ++j) {
            double s = 0.0;
            for (int i = 0; i < I; ++i)
                s += (double)X[r * I + i] * (double)W1[(size_t)i * H + j];
            y += (s > 0.0 ? s : 0.0) * (double)W2[j];
        }
        double e = y - (double)Y[r];
        se[r] = e * e;
    }
    double sse = 0.0;
    for (int64_t r = 0; r < n; ++r) sse += se[r];
    free(se);
    return sse / (double)n;
}

/* Per-row predictions (fp64) for sampled full-size checks: out[k] = Ypred of row rows[k]. */
void oracle_predict_rows(const float *X, const int64_t *rows, int64_t nrows, int I, int H,
                         const float *W1, const float *W2, double *out)
{
    for (int64_t k = 0; k < nrows; ++k) {
        const float *x = X + rows[k] * I;
        double y = 0.0;
        for (int j = 0; j < H; ++j) {
            double s = 0.0;
            for (int i = 0; i < I; ++i) s += (double)x[i] * (double)W1[(size_t)i * H + j];
            y += (s > 0.0 ? s : 0.0) * (double)W2[j];
        }
        out[k] = y;
    }
}

/*
 * Weight initialisation U(+-1/sqrt(fan_in)) -- the oracle-side restatement of the
 * counter-based generator that include/mlp.h documents for mlp_init_weights
 * (SURVEY.md 8(c) item 22).  Element index e runs over W1 row-major then W2:
 *   z = seed + 0x9E3779B97F4A7C15 * (e + 1)                   (mod 2^64)
 *   z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9 ; z = (z ^ (z >> 27)) * 0x94D049BB133111EB
 *   z =  z ^ (z >> 31)                                         (SplitMix64 finaliser)
 *   u = (z >> 40) * 2^-24  in [0,1) ;  w = (float)((2u - 1) * bound)
 * with bound = 1/sqrt(fan_in) in double, fan_in = I for W1 and H for W2.
 */
void oracle_init_weights(uint64_t seed, int I, int H, float *W1, float *W2)
{
    const double b1 = 1.0 / sqrt((double)I), b2 = 1.0 / sqrt((double)H);
    const uint64_t total = (uint64_t)I * H + (uint64_t)H;
    for (uint64_t e = 0; e < total; ++e) {
        uint64_t z = seed + 0x9E3779B97F4A7C15ULL * (e + 1);
        z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
        z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
        z = z ^ (z >> 31);
        double u = (double)(z >> 40) * (1.0 / 16777216.0);
        if (e < (uint64_t)I * H) W1[e] = (float)((2.0 * u - 1.0) * b1);
        else                     W2[e - (uint64_t)I * H] = (float)((2.0 * u - 1.0) * b2);
    }
}

int oracle_num_threads(void)
{
    int nt = 1;
#ifdef _OPENMP
    #pragma omp parallel
    {
        #pragma omp master
        nt = omp_get_num_threads();
    }
#endif
    return nt;
}
