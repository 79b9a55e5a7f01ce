/*
 * casgd_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, FP64 CPU restatement of one communication-avoiding SGD (CA-SGD)
 * outer iteration for generalized linear models, written from the paper's
 * definitions (arxiv/paper_2606_18463, /root/reference/PAPER.md). It exists so
 * the CUDA path has something independent to be compared with. It shares no
 * code, header, table or helper with paper_2606_18463_b200/csrc, and nothing
 * in the product path may call it (only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs do).
 *
 * Sign convention. The paper writes the residual delta = -dL/dr and updates
 * x <- x + (eta/b) Y^T delta (sec. 3.1, L135 Alg. 1 line 17).
 * This file uses u = dL/dr = -delta and x <- x - (eta/b) Y^T u, which is the
 * same algorithm (BASELINE.json:north_star uses the u-form).
 *
 * Readings of the paper taken here (DESIGN.md "Readings" lists them all):
 *   - Alg. 1 lines 8-15 (L121-L132) lost their if/else in extraction:
 *     j = 0: z^(0) = r_0;  j > 0: z^(j) = r_j + (eta/b) G_{j,<j} delta_hist.
 *   - alpha = eta/b everywhere, including the outer update (L126, L135, L180).
 *   - x enters the margin as its BF16 rounding (round-to-nearest-even), the
 *     update is applied to the un-rounded master x (L231, Table 1).
 *   - r, u stay in full precision (no BF16 cast of r: that cast only serves
 *     the AllReduce of L91, absent at P = 1).
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): finite differences of L
 * for l'; closed forms F(0); first block from x = 0; s = 1 == textbook
 * mini-batch SGD; Gram form == s sequential SGD steps (L176) to 1e-12; the
 * linear-loss recurrence == a LAPACK unit-lower-triangular solve and the
 * terminating Neumann series (L180); G symmetric PSD, rank <= n; brute-force
 * pure-Python loops on tiny inputs; BF16 helpers exhaustively against
 * torch.bfloat16.  The paper prints no worked numerical example of a step, so
 * no printed G, r, u or x exists to compare with: beyond those pins the
 * values are "parity unpinned" (DESIGN.md says the same).
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC (oracle/__init__.py does it).
 * OpenMP is used only to spread independent rows over cores; no summation is
 * split, blocked or reordered.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { LOSS_LOGISTIC = 0, LOSS_LINEAR = 1, LOSS_POISSON = 2 };

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---------------------------------------------------------------- BF16 --- */

/* BF16 is the upper 16 bits of an IEEE-754 binary32 (Table 3:
 * u_BF16 ~ 4e-3 = 2^-8). Widening is exact. */
double oracle_bf16_to_f64(uint16_t h)
{
    uint32_t w = (uint32_t)h << 16;
    float f;
    memcpy(&f, &w, sizeof f);
    return (double)f;
}

/* binary32 -> BF16, round to nearest, ties to even (reading 9: the paper is
 * silent on the rounding mode). NaN stays NaN (quiet). */
uint16_t oracle_f32_to_bf16(float f)
{
    uint32_t w;
    memcpy(&w, &f, sizeof w);
    if ((w & 0x7fffffffu) > 0x7f800000u)          /* NaN */
        return (uint16_t)((w >> 16) | 0x0040u);
    uint32_t keep_is_odd = (w >> 16) & 1u;
    w += 0x7fffu + keep_is_odd;                    /* RNE on the dropped 16 bits */
    return (uint16_t)(w >> 16);
}

/* binary64 -> BF16, round to nearest even, with no double rounding: take the
 * binary32 route as a first guess, then pick the nearest of that guess and
 * its two BF16 neighbours measured in binary64. */
uint16_t oracle_f64_to_bf16(double d)
{
    if (d != d) return 0x7fc0u;
    uint16_t guess = oracle_f32_to_bf16((float)d);
    if ((guess & 0x7fffu) == 0x7f80u) return guess;          /* +-inf */
    uint16_t best = guess;
    double best_err = fabs(oracle_bf16_to_f64(guess) - d);
    for (int step = -1; step <= 1; step += 2) {
        /* neighbour in magnitude order; the sign bit is carried along */
        uint16_t mag = guess & 0x7fffu, sign = guess & 0x8000u;
        if (step < 0 && mag == 0) continue;
        uint16_t cand = (uint16_t)(sign | (uint16_t)(mag + step));
        if ((cand & 0x7fffu) >= 0x7f80u) continue;
        double err = fabs(oracle_bf16_to_f64(cand) - d);
        if (err < best_err || (err == best_err && (cand & 1u) == 0 && (best & 1u) == 1)) {
            best = cand;
            best_err = err;
        }
    }
    return best;
}

/* ------------------------------------------------------- loss family ----- */

/* L(r, y), sec. 2.1:
 *   logistic log(1 + e^{-y r});  linear (r - y)^2 / 2;  Poisson e^r - y r.
 * The logistic form is evaluated as max(-t,0) + log1p(exp(-|t|)), t = y r,
 * which is the same function without overflow. */
double oracle_loss_value(double r, double y, int loss)
{
    switch (loss) {
    case LOSS_LOGISTIC: {
        double t = y * r;
        return (t < 0 ? -t : 0.0) + log1p(exp(-fabs(t)));
    }
    case LOSS_LINEAR:
        return 0.5 * (r - y) * (r - y);
    case LOSS_POISSON:
        return exp(r) - y * r;
    }
    return NAN;
}

/* u = dL/dr = -delta, with delta printed at PAPER.md:L59 sec. 3.1:
 *   logistic delta = y (1 - sigma(y r))  =>  u = -y / (1 + e^{y r})
 *   linear   delta = y - r               =>  u = r - y
 *   Poisson  delta = y - exp(r)          =>  u = e^r - y
 * The logistic branch is written so that exp never sees a positive argument. */
double oracle_lprime(double z, double y, int loss)
{
    switch (loss) {
    case LOSS_LOGISTIC: {
        double t = y * z;
        if (t >= 0) {
            double e = exp(-t);
            return -y * e / (1.0 + e);
        }
        return -y / (1.0 + exp(t));
    }
    case LOSS_LINEAR:
        return z - y;
    case LOSS_POISSON:
        return exp(z) - y;
    }
    return NAN;
}

/* F(x) = (1/m) sum_i L(a_i^T x, y_i). A holds BF16 bits, row
 * stride lda elements; x is the full-precision iterate (reading 17). */
double oracle_full_loss(const uint16_t *A, int64_t lda, const float *y, int64_t m, int32_t n,
                        const double *x, int loss)
{
    double total = 0.0;
#pragma omp parallel for reduction(+ : total) schedule(static)
    for (int64_t i = 0; i < m; ++i) {
        double r = 0.0;
        for (int32_t k = 0; k < n; ++k) r += oracle_bf16_to_f64(A[i * lda + k]) * x[k];
        total += oracle_loss_value(r, (double)y[i], loss);
    }
    return total / (double)m;
}

/* ------------------------------------------------------------ gather ----- */

/* Alg. 1 line 2 (L113): Y = A[I, :], y_I = y[I]. Y as doubles (exact widening),
 * and, when Y_bits != NULL, the raw BF16 bits for the bit-exact gather check. */
static int gather_rows(const uint16_t *A, int64_t lda, const float *y, int64_t m, int32_t n,
                       const int32_t *idx, int64_t sb, double *Y, double *yI, uint16_t *Y_bits)
{
    for (int64_t t = 0; t < sb; ++t) {
        int64_t row = idx[t];
        if (row < 0 || row >= m) return 1;
        for (int32_t k = 0; k < n; ++k) {
            uint16_t h = A[row * lda + k];
            Y[t * n + k] = oracle_bf16_to_f64(h);
            if (Y_bits) Y_bits[t * n + k] = h;
        }
        yI[t] = (double)y[row];
    }
    return 0;
}

/* x_hat: the vector the margin kernel sees. shadow = 1: BF16(x) (L231 "two
 * BF16 input conversions"); shadow = 0: x itself (all-FP32 Recipe A, L99). */
static void margin_input(const double *x, int32_t n, int shadow, double *x_hat)
{
    for (int32_t k = 0; k < n; ++k)
        x_hat[k] = shadow ? oracle_bf16_to_f64(oracle_f64_to_bf16(x[k])) : x[k];
}

/* ------------------------------------------------- O1: Gram form (Alg. 1) - */

/* One outer iteration exactly as Algorithm 1 states it,
 * at P = 1 (line 5's AllReduce is the identity):
 *   line 2   Y = A[I,:]
 *   line 3   r = Y x_hat
 *   line 4   G = Y Y^T                (the whole sb x sb matrix, no symmetry used)
 *   lines 6-15   for j = 0..s-1:  z_j = r_j - alpha * sum_{k<j} G_{jk} u_k ;
 *                                u_j = l'(z_j, y_{I_j})
 *   line 16  g = Y^T u
 *   line 17  x_out = x - alpha g      (master x, not x_hat)
 * Outputs (any may be NULL except x_out): Y_bits sb*n, G sb*sb, r, z, u (sb), g (n).
 * Returns 0, or 1 for an index outside [0, m), 2 for bad arguments / no memory. */
int oracle_outer_step_gram(const uint16_t *A, int64_t lda, const float *y, int64_t m, int32_t n,
                           const int32_t *idx, int32_t s, int32_t b, double eta, int loss, int shadow,
                           const double *x, uint16_t *Y_bits, double *G_out, double *r_out,
                           double *z_out, double *u_out, double *g_out, double *x_out)
{
    if (s < 1 || b < 1 || n < 1 || !x_out) return 2;
    const int64_t sb = (int64_t)s * b;
    const double alpha = eta / (double)b;
    double *Y = malloc(sizeof(double) * sb * n), *yI = malloc(sizeof(double) * sb);
    double *x_hat = malloc(sizeof(double) * n), *G = malloc(sizeof(double) * sb * sb);
    double *r = malloc(sizeof(double) * sb), *z = malloc(sizeof(double) * sb);
    double *u = malloc(sizeof(double) * sb), *g = malloc(sizeof(double) * n);
    int rc = 2;
    if (!Y || !yI || !x_hat || !G || !r || !z || !u || !g) goto done;
    rc = gather_rows(A, lda, y, m, n, idx, sb, Y, yI, Y_bits);
    if (rc) goto done;
    margin_input(x, n, shadow, x_hat);

    for (int64_t i = 0; i < sb; ++i) {                      /* line 3 */
        double acc = 0.0;
        for (int32_t k = 0; k < n; ++k) acc += Y[i * n + k] * x_hat[k];
        r[i] = acc;
    }
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < sb; ++i)                        /* line 4 */
        for (int64_t j = 0; j < sb; ++j) {
            double acc = 0.0;
            for (int32_t k = 0; k < n; ++k) acc += Y[i * n + k] * Y[j * n + k];
            G[i * sb + j] = acc;
        }
    for (int32_t j = 0; j < s; ++j)                         /* lines 6-15 */
        for (int32_t i = 0; i < b; ++i) {
            int64_t row = (int64_t)j * b + i;
            double corr = 0.0;
            for (int64_t t = 0; t < (int64_t)j * b; ++t) corr += G[row * sb + t] * u[t];
            z[row] = r[row] - alpha * corr;
            u[row] = oracle_lprime(z[row], yI[row], loss);
        }
    for (int32_t k = 0; k < n; ++k) {                       /* lines 16-17 */
        double acc = 0.0;
        for (int64_t t = 0; t < sb; ++t) acc += Y[t * n + k] * u[t];
        g[k] = acc;
        x_out[k] = x[k] - alpha * acc;
    }
    if (G_out) memcpy(G_out, G, sizeof(double) * sb * sb);
    if (r_out) memcpy(r_out, r, sizeof(double) * sb);
    if (z_out) memcpy(z_out, z, sizeof(double) * sb);
    if (u_out) memcpy(u_out, u, sizeof(double) * sb);
    if (g_out) memcpy(g_out, g, sizeof(double) * n);
done:
    free(Y); free(yI); free(x_hat); free(G); free(r); free(z); free(u); free(g);
    return rc;
}

/* Selected Gram entries G[i,j] = <Y_i, Y_j> for (i,j) = pairs[2p], pairs[2p+1]
 * (positions within the sampled block), for parity at sizes where the full
 * sb x sb matrix is too slow to form here. Also norms[t] = ||Y_t||_2 if given. */
int oracle_gram_entries(const uint16_t *A, int64_t lda, int64_t m, int32_t n, const int32_t *idx,
                        int64_t sb, const int64_t *pairs, int64_t npairs, double *out, double *norms)
{
    for (int64_t t = 0; t < sb; ++t)
        if (idx[t] < 0 || idx[t] >= m) return 1;
    for (int64_t p = 0; p < npairs; ++p) {
        const uint16_t *a = A + (int64_t)idx[pairs[2 * p]] * lda;
        const uint16_t *c = A + (int64_t)idx[pairs[2 * p + 1]] * lda;
        double acc = 0.0;
        for (int32_t k = 0; k < n; ++k) acc += oracle_bf16_to_f64(a[k]) * oracle_bf16_to_f64(c[k]);
        out[p] = acc;
    }
    if (norms)
        for (int64_t t = 0; t < sb; ++t) {
            const uint16_t *a = A + (int64_t)idx[t] * lda;
            double acc = 0.0;
            for (int32_t k = 0; k < n; ++k) acc += oracle_bf16_to_f64(a[k]) * oracle_bf16_to_f64(a[k]);
            norms[t] = sqrt(acc);
        }
    return 0;
}

/* -------------------------------------------- O2: sequential form (L176) -- */

/* "The exact CA-SGD block with parameter s is the composition of s mini-batch
 * SGD steps" (Assumption 5.6, L176; mini-batch SGD itself at L33). Started
 * from the margin input x_hat:
 *   v = x_hat; w = 0
 *   for j: z_j = Y_j v ; u_j = l'(z_j, y_{I_j}) ; d = alpha Y_j^T u_j ; v -= d ; w += d
 *   x_out = x - w
 * With shadow = 0 and s = 1 this is textbook mini-batch SGD. It never forms G:
 * sum_{k<j} G_{jk} u_k = Y_j (sum_{k<j} Y_k^T u_k). */
static int seq_step(const uint16_t *A, int64_t lda, const float *y, int64_t m, int32_t n,
                    const int32_t *idx, int32_t s, int32_t b, double alpha, int loss, int shadow,
                    double *x, double *Yj, double *yI, double *v, double *w, double *z_out, double *u_out,
                    double *uj)
{
    margin_input(x, n, shadow, v);
    for (int32_t k = 0; k < n; ++k) w[k] = 0.0;
    for (int32_t j = 0; j < s; ++j) {
        int rc = gather_rows(A, lda, y, m, n, idx + (int64_t)j * b, b, Yj, yI, NULL);
        if (rc) return rc;
#pragma omp parallel for schedule(static) if ((int64_t)b * n > 65536)
        for (int32_t i = 0; i < b; ++i) {
            double acc = 0.0;
            for (int32_t k = 0; k < n; ++k) acc += Yj[(int64_t)i * n + k] * v[k];
            uj[i] = oracle_lprime(acc, yI[i], loss);
            if (z_out) z_out[(int64_t)j * b + i] = acc;
            if (u_out) u_out[(int64_t)j * b + i] = uj[i];
        }
#pragma omp parallel for schedule(static) if ((int64_t)b * n > 65536)
        for (int32_t k = 0; k < n; ++k) {
            double acc = 0.0;
            for (int32_t i = 0; i < b; ++i) acc += Yj[(int64_t)i * n + k] * uj[i];
            double d = alpha * acc;
            v[k] -= d;
            w[k] += d;
        }
    }
    for (int32_t k = 0; k < n; ++k) x[k] -= w[k];
    return 0;
}

/* n_outer consecutive outer iterations in the sequential form, x updated in
 * place; idx holds n_outer*s*b indices. With n_outer = 1 and z/u given this is
 * O2 for one step; with many steps it is the trajectory oracle (master x in
 * binary64, x_hat = BF16(x) refreshed once per outer step when shadow = 1). */
int oracle_train_seq(const uint16_t *A, int64_t lda, const float *y, int64_t m, int32_t n,
                     const int32_t *idx, int64_t n_outer, int32_t s, int32_t b, double eta, int loss,
                     int shadow, double *x, double *z_out, double *u_out)
{
    if (s < 1 || b < 1 || n < 1 || n_outer < 0) return 2;
    double *Yj = malloc(sizeof(double) * (size_t)b * n), *yI = malloc(sizeof(double) * b);
    double *v = malloc(sizeof(double) * n), *w = malloc(sizeof(double) * n), *uj = malloc(sizeof(double) * b);
    int rc = 2;
    if (Yj && yI && v && w && uj) {
        rc = 0;
        const int64_t sb = (int64_t)s * b;
        for (int64_t h = 0; h < n_outer && !rc; ++h)
            rc = seq_step(A, lda, y, m, n, idx + h * sb, s, b, eta / (double)b, loss, shadow, x, Yj, yI, v, w,
                          z_out ? z_out + h * sb : NULL, u_out ? u_out + h * sb : NULL, uj);
    }
    free(Yj); free(yI); free(v); free(w); free(uj);
    return rc;
}

/* n_outer consecutive outer iterations in the Gram form (O1), x in place;
 * used to check O1 == O2 over a whole trajectory on the tiny config and as the
 * timed "what the GPU computes" CPU baseline. */
int oracle_train_gram(const uint16_t *A, int64_t lda, const float *y, int64_t m, int32_t n,
                      const int32_t *idx, int64_t n_outer, int32_t s, int32_t b, double eta, int loss,
                      int shadow, double *x)
{
    double *x_next = malloc(sizeof(double) * n);
    if (!x_next) return 2;
    int rc = 0;
    const int64_t sb = (int64_t)s * b;
    for (int64_t h = 0; h < n_outer && !rc; ++h) {
        rc = oracle_outer_step_gram(A, lda, y, m, n, idx + h * sb, s, b, eta, loss, shadow, x, NULL, NULL, NULL,
                                    NULL, NULL, NULL, x_next);
        if (!rc) memcpy(x, x_next, sizeof(double) * n);
    }
    free(x_next);
    return rc;
}
