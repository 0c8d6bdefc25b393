/*
 * phx_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, one-element-at-a-time CPU statement of what the hot path
 * computes (the paper names the states — "Adam optimizer
 * states (first and second moments, together with the FP32 master copy)",
 * PAPER.md:270, "ZeRO-2 distributed optimizer", PAPER.md:272 — but never
 * prints the update, so the sequence below is DESIGN.md reading R1).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * `--impl reference` leg may call this.  It shares no code with the CUDA
 * path under paper_2607_01646_b200/csrc and neither includes the other.
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fno-fast-math -fopenmp -shared -fPIC
 *   -ffp-contract=off : every + - * / below is ONE IEEE-754 binary32 (or
 *                       binary64) operation, round-to-nearest-even, no FMA.
 *   x86-64 SSE2 arithmetic does not flush denormals and has correctly rounded
 *   sqrtf and division.
 * OpenMP only splits the element loop into contiguous ranges (the update is
 * elementwise, so the thread count cannot change a single bit); it exists so
 * that bench.py can time the oracle on all host cores.
 *
 * Pins (tests/test_oracle_pins.py): closed forms from m=v=0, constant-gradient
 * trajectories, zero-gradient decay, lr=0 / wd=0 degenerate cases, sign
 * symmetry, the |update| <= 1.165*lr bound, exact rational evaluation on tiny
 * inputs, torch.optim.AdamW (CPU) as a library special case, a float64 shadow,
 * torch's bf16 cast for the rounding, hand-computable norms for the clip.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <string.h>

/* ---- bf16 <-> fp32 (reading R1, last line of the canonical sequence) ------ */

static float widen_bf16(uint16_t h)
{
    uint32_t u = (uint32_t)h << 16; /* exact: bf16 is the top half of binary32 */
    float f;
    memcpy(&f, &u, 4);
    return f;
}

/* round-to-nearest-even on the low 16 bits; NaN is outside the tested domain */
uint16_t phx_oracle_rne_bf16(float x)
{
    uint32_t u;
    memcpy(&u, &x, 4);
    u += 0x7FFFu + ((u >> 16) & 1u);
    return (uint16_t)(u >> 16);
}

/* ---- derived scalars (reading R6): double on the host, rounded once ------- */

/* beta^t by LSB-first square-and-multiply in double (deterministic, no libm pow) */
static double pow_sqmul(double b, uint64_t t)
{
    double r = 1.0;
    while (t) {
        if (t & 1u)
            r = r * b;
        b = b * b;
        t >>= 1;
    }
    return r;
}

/* out = {decay, omb1, omb2, ss, sbc2}; t = 1-based step (reading R3) */
void phx_oracle_scalars(float lr, float beta1, float beta2, float eps, float wd,
                        uint64_t t, float out[5])
{
    (void)eps;
    double dlr = (double)lr, db1 = (double)beta1, db2 = (double)beta2, dwd = (double)wd;
    out[0] = (float)(1.0 - dlr * dwd);                    /* decay = 1 - lr*wd        */
    out[1] = (float)(1.0 - db1);                          /* omb1  = 1 - beta1        */
    out[2] = (float)(1.0 - db2);                          /* omb2  = 1 - beta2        */
    out[3] = (float)(dlr / (1.0 - pow_sqmul(db1, t)));    /* ss    = lr/(1-beta1^t)   */
    out[4] = (float)sqrt(1.0 - pow_sqmul(db2, t));        /* sbc2  = sqrt(1-beta2^t)  */
}

/* ---- a3: one AdamW step over a shard, canonical sequence (reading R1) ------
 *   g   = widen(g_bf16) * coef          coef = clip coefficient, 1.0f when off
 *   p1  = p * decay
 *   m'  = (beta1*m) + (omb1*g)
 *   v'  = (beta2*v) + (omb2*(g*g))
 *   d   = (sqrt(v') / sbc2) + eps
 *   p'  = p1 - (ss * (m'/d))
 *   p16 = RNE_bf16(p')
 * volatile temporaries are not needed: -ffp-contract=off forbids fusing. */
void phx_oracle_adamw_step(float *p, float *m, float *v, const uint16_t *g_bf16,
                           uint16_t *p16, size_t n, float lr, float beta1,
                           float beta2, float eps, float wd, uint64_t t, float coef,
                           int nthreads)
{
    float sc[5];
    phx_oracle_scalars(lr, beta1, beta2, eps, wd, t, sc);
    const float decay = sc[0], omb1 = sc[1], omb2 = sc[2], ss = sc[3], sbc2 = sc[4];
    (void)nthreads;
#pragma omp parallel for schedule(static) num_threads(nthreads > 0 ? nthreads : 1)
    for (ptrdiff_t i = 0; i < (ptrdiff_t)n; ++i) {
        float g = widen_bf16(g_bf16[i]);
        g = g * coef;
        float p1 = p[i] * decay;
        float a = beta1 * m[i];
        float b = omb1 * g;
        float mn = a + b;
        float gg = g * g;
        float c = beta2 * v[i];
        float e = omb2 * gg;
        float vn = c + e;
        float s = sqrtf(vn);
        float q = s / sbc2;
        float d = q + eps;
        float r = mn / d;
        float u = ss * r;
        float pn = p1 - u;
        p[i] = pn;
        m[i] = mn;
        v[i] = vn;
        p16[i] = phx_oracle_rne_bf16(pn);
    }
}

/* ---- a1: sum of squares and clip coefficient (reading R7) ------------------
 * Each square of a widened bf16 is exact in double (16 significant bits); the
 * running sum is kept in long double (x87, 64-bit significand) and rounded to
 * double once.  tests pin it to math.fsum (the exactly rounded sum). */
double phx_oracle_sumsq(const uint16_t *g_bf16, size_t n)
{
    long double s = 0.0L;
    for (size_t i = 0; i < n; ++i) {
        double g = (double)widen_bf16(g_bf16[i]);
        s += (long double)(g * g);
    }
    return (double)s;
}

/* coef = fp32( min(1, max_norm / (sqrt(S) + 1e-6)) ), all in double until the end */
float phx_oracle_clip_coef(double sumsq, float max_norm)
{
    double norm = sqrt(sumsq);
    double c = (double)max_norm / (norm + 1e-6);
    if (c > 1.0)
        c = 1.0;
    return (float)c;
}

/* ---- regeneration of the bf16 copy at restore (reading R9) ---------------- */
void phx_oracle_regen_bf16(const float *p, uint16_t *p16, size_t n)
{
    for (size_t i = 0; i < n; ++i)
        p16[i] = phx_oracle_rne_bf16(p[i]);
}

/* ==== SURVEY.md §8(f2): the paper's own precision and per-tensor decay groups ====
 *
 * "all parameters, main gradients and optimizer states (Adam moments together with the
 * FP32 master copy) use torch.float32 ... BF16 and FP16 disabled": the
 * gradients arrive as binary32 and there is no bf16 model-parameter copy.  The sequence
 * is reading R1 unchanged except for its first line (g = g_f32 * coef, no widening) and
 * its last (no RNE_bf16).  g*g is now a rounded binary32 product (24-bit significands).
 *
 * Decay groups (reading R5b): a tensor flagged "no decay" (biases, norm
 * weights — the usual AdamW parameter groups) takes weight decay 0, i.e. decay = 1.0f
 * for its elements; p * 1.0f is exact, so its trajectory is bit-identical to a wd = 0 run.
 *
 * One general routine: exactly one of g_bf16 / g_f32 is non-NULL; p16 may be NULL (no
 * bf16 copy); no_decay may be NULL (uniform decay), else one byte per element. */
void phx_oracle_adamw_step_ex(float *p, float *m, float *v, const uint16_t *g_bf16,
                              const float *g_f32, uint16_t *p16, const uint8_t *no_decay,
                              size_t n, float lr, float beta1, float beta2, float eps,
                              float wd, uint64_t t, float coef, int nthreads)
{
    float sc[5];
    phx_oracle_scalars(lr, beta1, beta2, eps, wd, t, sc);
    const float decay = sc[0], omb1 = sc[1], omb2 = sc[2], ss = sc[3], sbc2 = sc[4];
    (void)nthreads;
#pragma omp parallel for schedule(static) num_threads(nthreads > 0 ? nthreads : 1)
    for (ptrdiff_t i = 0; i < (ptrdiff_t)n; ++i) {
        float g = g_f32 ? g_f32[i] : widen_bf16(g_bf16[i]);
        g = g * coef;
        float dk = (no_decay && no_decay[i]) ? 1.0f : decay;
        float p1 = p[i] * dk;
        float a = beta1 * m[i];
        float b = omb1 * g;
        float mn = a + b;
        float gg = g * g;
        float c = beta2 * v[i];
        float e = omb2 * gg;
        float vn = c + e;
        float s = sqrtf(vn);
        float q = s / sbc2;
        float d = q + eps;
        float r = mn / d;
        float u = ss * r;
        float pn = p1 - u;
        p[i] = pn;
        m[i] = mn;
        v[i] = vn;
        if (p16)
            p16[i] = phx_oracle_rne_bf16(pn);
    }
}

/* Sum of squares of binary32 gradients: each square is exact in double (48 significant
 * bits); the running sum is long double, rounded to double once (as phx_oracle_sumsq). */
double phx_oracle_sumsq_f32(const float *g, size_t n)
{
    long double s = 0.0L;
    for (size_t i = 0; i < n; ++i) {
        double x = (double)g[i];
        s += (long double)(x * x);
    }
    return (double)s;
}

/* ==== SURVEY.md §8(f4), second half: the gradient producer's epilogue ======================
 *
 * "single-pass fusion of the sum-of-squares with the previous step's epilogue" (SURVEY.md §8(f),
 * row f4).  What precedes a1 in the ZeRO-2 distributed optimizer is the
 * reduce-scatter of the binary32 main gradients ("main gradients ... torch.float32")
 * and their averaging / cast to the optimizer's gradient dtype.  DESIGN.md reading R34:
 *
 *   h_i   = g32_i * scale          one binary32 multiply (scale = 1/(dp_size*microbatches); 1.0f is exact)
 *   g16_i = RNE_bf16(h_i)          the same integer rounding as the last line of reading R1
 *   S     = sum_i widen(g16_i)^2   of the ROUNDED values — it must equal what a1 (phx_oracle_sumsq)
 *                                  computes from the bf16 gradients the optimizer then reads
 *
 * Plain statement: one loop, the rounding first, the square of the rounded value second, the
 * running sum in long double rounded to double once (exactly as phx_oracle_sumsq). */
double phx_oracle_grads_finalize(const float *g32, float scale, uint16_t *g_bf16, size_t n)
{
    long double s = 0.0L;
    for (size_t i = 0; i < n; ++i) {
        float h = g32[i] * scale;
        uint16_t b = phx_oracle_rne_bf16(h);
        g_bf16[i] = b;
        double w = (double)widen_bf16(b);
        s += (long double)(w * w);
    }
    return (double)s;
}
