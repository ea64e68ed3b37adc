/*
 * ozaki2_oracle.c -- plain, slow, CPU-only ORACLE for DGEMM emulated by Ozaki scheme II
 * with its three scaling modes (accurate / original fast / revised fast).
 *
 * THIS FILE IS TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code,
 * header, table or constant generator with the CUDA library under
 * paper_2606_29129_b200/csrc/ and never includes anything from there.
 *
 * It follows the paper (/root/reference/PAPER.md, cited as P:<line>) step by step, in
 * the paper's order and notation, with wide integers instead of any blocking or fusion:
 *
 *   O1  constants            Step 1 P:90, eq.(14), P'_accu P:141-143,
 *                            P'_fast P:193-195, P'_prop P:326-328, delta eq.(6)
 *   O2  row/column statistics  max and rounded-up sum of squares, Alg.1/2 "Require" lines
 *                            P:174-176; reading R2 of DESIGN.md (integer sum)
 *   O3  exponents            Alg.1 P:182-184 (eq.11/12), Alg.2 P:336-338 (eq.17/18),
 *                            accurate mode P:123-157 (eq.4-9, reading G3 of DESIGN.md)
 *   O4  truncation           a' = trunc(mu_i a), Step 2 P:91-95
 *   O5  residues             rmod(A', p_l) as INT8, P:70, P:103, P:113 (reading R5)
 *   O6  per-modulus products INT8 x INT8 -> wide accumulate, then mod p_l, eq.(2)
 *   O7  CRT                  C' = sum P_l q_l U_l, C'' = rmod(C', P), eq.(2)(3)
 *   O8  exact product        Z = A'B' and sum |a'||b'| in 256-bit integers; condition (1) P:99
 *   O9  unscale, alpha/beta  Step 4 P:109-111 (readings R8, R9)
 *   O10 reports              effective bit width P:207-213, double-double reference P:268
 *
 * Precision: integer stages are exact (own 256-bit two's-complement type); the FP32
 * steps the paper fixes (single_up / single_down) are single IEEE operations done
 * under fesetround(); the final C is FP64 as in the paper.
 *
 * Parity pins (tests/test_oracle_*.py, -m "not gpu"): eq.(14) list and CRT identities,
 * constants against 400-bit mpmath, the paper's all-ones worked example,
 * closed forms on all-ones inputs, exact-rational truncation, brute-force CRT on tiny
 * integer matrices against Python integers, condition (1) for the revised mode,
 * scale invariance, textbook special cases for the final C.
 * No function here is "parity unpinned".
 *
 * Build: gcc -O2 -fopenmp -frounding-math -fno-fast-math -shared -fPIC (oracle/build.py).
 */
#include <fenv.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef __int128 i128;
typedef unsigned __int128 u128;

/* ------------------------------------------------------------------------------------ */
/* 256-bit two's-complement integer, little-endian 64-bit words                          */
/* ------------------------------------------------------------------------------------ */
typedef struct { uint64_t w[4]; } wint;

static wint w_zero(void) { wint r; memset(&r, 0, sizeof r); return r; }

static wint w_from_u64(uint64_t v) { wint r = w_zero(); r.w[0] = v; return r; }

static int w_isneg(wint a) { return (int)(a.w[3] >> 63); }

static int w_iszero(wint a) { return (a.w[0] | a.w[1] | a.w[2] | a.w[3]) == 0; }

static wint w_add(wint a, wint b)
{
    wint r;
    unsigned carry = 0;
    for (int i = 0; i < 4; i++) {
        u128 s = (u128)a.w[i] + b.w[i] + carry;
        r.w[i] = (uint64_t)s;
        carry = (unsigned)(s >> 64);
    }
    return r;
}

static wint w_not(wint a)
{
    wint r;
    for (int i = 0; i < 4; i++) r.w[i] = ~a.w[i];
    return r;
}

static wint w_neg(wint a) { return w_add(w_not(a), w_from_u64(1)); }

static wint w_sub(wint a, wint b) { return w_add(a, w_neg(b)); }

static wint w_abs(wint a) { return w_isneg(a) ? w_neg(a) : a; }

/* signed comparison: -1, 0, +1 */
static int w_cmp(wint a, wint b)
{
    int na = w_isneg(a), nb = w_isneg(b);
    if (na != nb) return na ? -1 : 1;
    for (int i = 3; i >= 0; i--) {
        if (a.w[i] < b.w[i]) return -1;
        if (a.w[i] > b.w[i]) return 1;
    }
    return 0;
}

/* logical shift left by 0 <= n < 256 */
static wint w_shl(wint a, int n)
{
    wint r = w_zero();
    int ws = n / 64, bs = n % 64;
    for (int i = 3; i >= ws; i--) {
        uint64_t v = a.w[i - ws] << bs;
        if (bs && i - ws - 1 >= 0) v |= a.w[i - ws - 1] >> (64 - bs);
        r.w[i] = v;
    }
    return r;
}

/* non-negative a times a 64-bit unsigned factor (caller guarantees no overflow) */
static wint w_mul_u64(wint a, uint64_t b)
{
    wint r;
    uint64_t carry = 0;
    for (int i = 0; i < 4; i++) {
        u128 t = (u128)a.w[i] * b + carry;
        r.w[i] = (uint64_t)t;
        carry = (uint64_t)(t >> 64);
    }
    return r;
}

/* exact signed product of two 128-bit integers */
static wint w_mul_i128(i128 a, i128 b)
{
    int neg = (a < 0) != (b < 0);
    u128 ua = a < 0 ? (u128)0 - (u128)a : (u128)a;
    u128 ub = b < 0 ? (u128)0 - (u128)b : (u128)b;
    uint64_t x[2] = { (uint64_t)ua, (uint64_t)(ua >> 64) };
    uint64_t y[2] = { (uint64_t)ub, (uint64_t)(ub >> 64) };
    uint64_t acc[4] = { 0, 0, 0, 0 };
    for (int i = 0; i < 2; i++) {
        uint64_t carry = 0;
        for (int j = 0; j < 2; j++) {
            u128 t = (u128)x[i] * y[j] + acc[i + j] + carry;
            acc[i + j] = (uint64_t)t;
            carry = (uint64_t)(t >> 64);
        }
        acc[i + 2] += carry;
    }
    wint r;
    memcpy(r.w, acc, sizeof acc);
    return neg ? w_neg(r) : r;
}

/* number of significant bits of a non-negative value (0 for zero) */
static int w_bitlen(wint a)
{
    for (int i = 3; i >= 0; i--)
        if (a.w[i]) return 64 * i + 64 - __builtin_clzll(a.w[i]);
    return 0;
}

/* bit t of a non-negative value */
static int w_bit(wint a, int t) { return (t < 0 || t >= 256) ? 0 : (int)((a.w[t / 64] >> (t % 64)) & 1); }

/* a mod p for non-negative a, 2 <= p <= 2^16 */
static unsigned w_mod_small(wint a, unsigned p)
{
    u128 r = 0;
    for (int i = 3; i >= 0; i--) r = ((r << 64) | a.w[i]) % p;
    return (unsigned)r;
}

/* RN_64(v * 2^sh): the correctly rounded double (ties to even) of the exact value,
 * with a single rounding also when the result is subnormal; +-inf on overflow.
 * (reading R8: "RN_64 of the exact integer, then exact power-of-two scaling") */
static double w_to_double_scaled(wint v, long sh)
{
    if (w_iszero(v)) return 0.0;
    int neg = w_isneg(v);
    wint a = w_abs(v);
    int t = w_bitlen(a) - 1;               /* a in [2^t, 2^(t+1)) */
    long E = (long)t + sh;                 /* value in [2^E, 2^(E+1)) */
    long qe = E - 52;                      /* exponent of the last kept bit */
    if (qe < -1074) qe = -1074;            /* subnormal quantum */
    long r = qe - sh;                      /* bits of a dropped below the quantum */
    uint64_t q;                            /* kept integer: value ~ q * 2^qe */
    if (r <= 0) {
        /* nothing dropped: a has at most 53 bits here */
        q = a.w[0] << (-r);
    } else if (r > 256) {
        q = 0;
    } else {
        /* q = floor(a / 2^r), then round to nearest, ties to even */
        q = 0;
        for (int b = 0; b < 54; b++) q |= (uint64_t)w_bit(a, (int)r + b) << b;
        int half = w_bit(a, (int)r - 1);
        int sticky = 0;
        for (int b = 0; b < (int)r - 1 && !sticky; b++) sticky = w_bit(a, b);
        if (half && (sticky || (q & 1))) q += 1;
    }
    double d = ldexp((double)q, (int)qe);  /* q <= 2^53: exact; ldexp overflows to inf */
    return neg ? -d : d;
}

/* ------------------------------------------------------------------------------------ */
/* FP32 operations with the rounding direction the paper writes                   */
/* ------------------------------------------------------------------------------------ */
static float f32_add_dir(float a, float b, int dir)
{
    volatile float x = a, y = b, r;
    int old = fegetround();
    fesetround(dir);
    r = x + y;
    fesetround(old);
    return r;
}
static float f32_sub_dir(float a, float b, int dir)
{
    volatile float x = a, y = b, r;
    int old = fegetround();
    fesetround(dir);
    r = x - y;
    fesetround(old);
    return r;
}
static float f32_mul_dir(float a, float b, int dir)
{
    volatile float x = a, y = b, r;
    int old = fegetround();
    fesetround(dir);
    r = x * y;
    fesetround(old);
    return r;
}
static float f32_fma_dir(float a, float b, float c, int dir)
{
    volatile float x = a, y = b, z = c, r;
    int old = fegetround();
    fesetround(dir);
    r = fmaf(x, y, z);
    fesetround(old);
    return r;
}
/* smallest float >= v (v a non-negative integer below 2^64) */
static float f32_from_u64_up(uint64_t v)
{
    float f = (float)v;                               /* round to nearest */
    if ((long double)f < (long double)v) f = nextafterf(f, INFINITY);
    return f;
}

/* exports of the primitives, so that the tests can pin them against exact rationals */
float oz2o_f32_add(float a, float b, int up) { return f32_add_dir(a, b, up ? FE_UPWARD : FE_DOWNWARD); }
float oz2o_f32_sub(float a, float b, int up) { return f32_sub_dir(a, b, up ? FE_UPWARD : FE_DOWNWARD); }
float oz2o_f32_mul(float a, float b, int up) { return f32_mul_dir(a, b, up ? FE_UPWARD : FE_DOWNWARD); }
float oz2o_f32_fma(float a, float b, float c, int up) { return f32_fma_dir(a, b, c, up ? FE_UPWARD : FE_DOWNWARD); }
float oz2o_f32_from_u64_up(uint64_t v) { return f32_from_u64_up(v); }

/* ------------------------------------------------------------------------------------ */
/* LOG2F: stand-in for __log2f on [1,2] (reading R3): the correctly rounded value        */
/* RN_32(log2 x).  |LOG2F(x) - log2 x| <= u32 < 4 u32, so every bound of P:145    */
/* holds.  Evaluated in 64-bit-mantissa long double, rounded once.                       */
/* ------------------------------------------------------------------------------------ */
float oz2o_log2f(float x) { return (float)log2l((long double)x); }
void oz2o_log2f_array(const float *x, float *y, long n) { for (long t = 0; t < n; t++) y[t] = oz2o_log2f(x[t]); }

/* ------------------------------------------------------------------------------------ */
/* O1 constants                                                                          */
/* ------------------------------------------------------------------------------------ */
#define OZ_MAX_MODULI 20
/* eq. (14); the first N are used (reading R1) */
static const int OZ_MODULI[OZ_MAX_MODULI] = { 256, 255, 253, 251, 247, 241, 239, 233, 229, 227,
                                              223, 217, 211, 199, 197, 193, 191, 181, 179, 173 };

typedef struct {
    int N;
    int p[OZ_MAX_MODULI];
    int q[OZ_MAX_MODULI];        /* q_l = P_l^{-1} mod p_l          (Step 1) */
    wint P;                      /* prod p_l                                        */
    wint Pl[OZ_MAX_MODULI];      /* P_l = P / p_l                                   */
    wint w[OZ_MAX_MODULI];       /* w_l = P_l q_l (< P)  weight of eq. (2)   */
    float Pprop, Paccu, Pfast;
    float delta;                 /* eq. (6)                                  */
} oz_consts;

static long double w_to_long_double(wint a) /* a >= 0; nearest up to one rounding per word */
{
    long double r = 0.0L;
    for (int i = 3; i >= 0; i--) r = r * 18446744073709551616.0L + (long double)a.w[i];
    return r;
}

static float round_down_to_f32(long double x)
{
    float f = (float)x;
    if ((long double)f > x) f = nextafterf(f, -INFINITY);
    return f;
}
static float round_up_to_f32(long double x)
{
    float f = (float)x;
    if ((long double)f < x) f = nextafterf(f, INFINITY);
    return f;
}

static int oz_make_consts(int N, oz_consts *c)
{
    if (N < 2 || N > OZ_MAX_MODULI) return -1;
    memset(c, 0, sizeof *c);
    c->N = N;
    c->P = w_from_u64(1);
    for (int l = 0; l < N; l++) {
        c->p[l] = OZ_MODULI[l];
        c->P = w_mul_u64(c->P, (uint64_t)c->p[l]);
    }
    for (int l = 0; l < N; l++) {
        wint Pl = w_from_u64(1);
        for (int j = 0; j < N; j++)
            if (j != l) Pl = w_mul_u64(Pl, (uint64_t)c->p[j]);
        c->Pl[l] = Pl;
        unsigned r = w_mod_small(Pl, (unsigned)c->p[l]);
        int q = -1;
        for (int t = 1; t < c->p[l]; t++)
            if ((r * (unsigned)t) % (unsigned)c->p[l] == 1u) { q = t; break; }
        if (q < 0) return -2; /* not coprime */
        c->q[l] = q;
        c->w[l] = w_mul_u64(Pl, (uint64_t)q);
    }
    /* P' constants: single_down(log2(P-1)/2 - c) */
    long double l2 = log2l(w_to_long_double(w_sub(c->P, w_from_u64(1))));
    c->Pprop = round_down_to_f32(l2 / 2.0L - 0.5L);
    c->Paccu = c->Pprop;
    c->Pfast = round_down_to_f32(l2 / 2.0L - 1.5L);
    /* delta = single_up(0.5 / (1 - 4 u32)), u32 = 2^-24 */
    c->delta = round_up_to_f32(0.5L / (1.0L - 4.0L * ldexpl(1.0L, -24)));
    return 0;
}

/* Export.  P_words: 4 x u64; w_words: N x 4 x u64 (little-endian). */
int oz2o_constants(int N, int *p, int *q, uint64_t *P_words, uint64_t *w_words,
                   float *Pprop, float *Pfast, float *delta)
{
    oz_consts c;
    int rc = oz_make_consts(N, &c);
    if (rc) return rc;
    for (int l = 0; l < N; l++) {
        p[l] = c.p[l];
        q[l] = c.q[l];
        memcpy(w_words + 4 * l, c.w[l].w, 32);
    }
    memcpy(P_words, c.P.w, 32);
    *Pprop = c.Pprop;
    *Pfast = c.Pfast;
    *delta = c.delta;
    return 0;
}

/* ------------------------------------------------------------------------------------ */
/* helpers on FP64 inputs                                                                */
/* ------------------------------------------------------------------------------------ */
/* |v| = M * 2^q with M an integer, 2^52 <= M < 2^53 (also for subnormals); v != 0 */
static void decompose(double v, uint64_t *M, int *q)
{
    int e;
    double m = frexp(fabs(v), &e);          /* m in [0.5, 1) */
    *M = (uint64_t)ldexp(m, 53);            /* exact */
    *q = e - 53;
}

/* floor(log2 |v|), v != 0, "from the exponent field", true value for subnormals */
static int floor_log2_abs(double v)
{
    int e;
    (void)frexp(fabs(v), &e);
    return e - 1;
}

/* element (r, c) of a column-major matrix */
#define CM(ptr, ld, r, c) ((ptr)[(size_t)(r) + (size_t)(c) * (size_t)(ld)])

/* ------------------------------------------------------------------------------------ */
/* O2 statistics of one vector v[0..k) with stride `st`                                  */
/*   E    = floor(log2 max|v_h|)                                                         */
/*   Sfix = sum_h ceil(2^SQ (v_h / 2^E)^2)   (exact integers; reading R2: an order-       */
/*          independent "rounding-up" evaluation of the sum of squares)     */
/*   SQ = 44 for k <= 2^17 (the range of P:113).  For longer k (blocked products)  */
/*   the fixed-point position drops by 2 for every factor 4 of k so that Sfix < 2^64:      */
/*   SQ = 44 - 2 ceil((ceil(log2 k) - 17) / 2)   (reading R2b of DESIGN.md)                */
/* returns 0 if the vector is all zero                                                   */
/* ------------------------------------------------------------------------------------ */
static int sq_shift(long k)
{
    int lg = 0;
    while (((long)1 << lg) < k) lg++;       /* ceil(log2 k) */
    int extra = lg > 17 ? lg - 17 : 0;
    return 44 - 2 * ((extra + 1) / 2);
}

static int vec_stats(const double *v, size_t st, long k, int *E_out, uint64_t *Sfix_out)
{
    const int SQ = sq_shift(k);
    double vmax = 0.0;
    for (long h = 0; h < k; h++) {
        double a = fabs(v[(size_t)h * st]);
        if (a > vmax) vmax = a;
    }
    if (!(vmax > 0.0)) { *E_out = 0; *Sfix_out = 0; return 0; }
    int E = floor_log2_abs(vmax);
    uint64_t S = 0;
    for (long h = 0; h < k; h++) {
        double a = v[(size_t)h * st];
        if (a == 0.0) continue;
        uint64_t M; int q;
        decompose(a, &M, &q);
        /* 2^SQ (a/2^E)^2 = M^2 * 2^(2(q-E)+SQ); M^2 < 2^106 */
        u128 M2 = (u128)M * M;
        long sh = 2L * (q - E) + SQ;        /* <= -60 because |a| < 2^(E+1) */
        uint64_t T;
        if (sh >= 0) return -1;             /* cannot happen */
        if (-sh >= 128) T = 1;              /* 0 < value < 1 */
        else {
            u128 fl = M2 >> (-sh);
            u128 rem = M2 & ((((u128)1) << (-sh)) - 1);
            T = (uint64_t)fl + (rem != 0);
        }
        S += T;                             /* <= k * 2^(SQ+2) <= 2^63 */
    }
    *E_out = E;
    *Sfix_out = S;
    return 1;
}

/* Alg.1 / Alg.2 on the statistics of one row or column (O3, modes 1 and 2).
 * F = RU_32(Sfix), shat = floor(log2 F) - SQ, x = F / 2^floor(log2 F), L = LOG2F(x). */
static int exponent_fast_or_prop(int mode, const oz_consts *c, int E, uint64_t Sfix, int SQ)
{
    float F = f32_from_u64_up(Sfix);
    int fe;
    float fm = frexpf(F, &fe);              /* F = fm 2^fe, fm in [0.5,1) */
    int shat = (fe - 1) - SQ;
    float x = 2.0f * fm;                    /* in [1,2), exact */
    float L = oz2o_log2f(x);
    if (mode == 2) {
        /* Algorithm 2, on the normalised sum (reading R11), then -E:
         *   t = single_up(0.5 * __log2f(a_norm/2^s) + 2 u32)
         *   w = single_down(P'_prop - 0.5 s)
         *   return floor(w - t)                                                        */
        float t = f32_fma_dir(0.5f, L, ldexpf(1.0f, -23), FE_UPWARD);
        float w = f32_sub_dir(c->Pprop, 0.5f * (float)shat, FE_DOWNWARD);
        float d = f32_sub_dir(w, t, FE_DOWNWARD);
        return (int)floorf(d) - E;
    } else {
        /* Algorithm 1, on the raw sum  a_norm = Shat * 2^(2E):
         *   s = floor(log2 a_norm)
         *   t = single_up(delta * (__log2f(a_norm/2^s) + s))
         *   return floor(P'_fast - max(1.0, t)) - floor(log2 a_max)                      */
        int s = shat + 2 * E;
        float inner = f32_add_dir(L, (float)s, FE_UPWARD);
        float t = f32_mul_dir(c->delta, inner, FE_UPWARD);
        float mx = t > 1.0f ? t : 1.0f;
        float d = f32_sub_dir(c->Pfast, mx, FE_DOWNWARD);
        return (int)floorf(d) - E;
    }
}

/* eq. (8)/(9) with reading G3: e = g + floor(P'_accu - delta * log2~(M)), g = 5 - E,
 * log2~ of eq. (7); M := max(M, 1) (reading R4). */
static int exponent_accurate(const oz_consts *c, int E, int64_t M)
{
    if (M < 1) M = 1;
    float F = f32_from_u64_up((uint64_t)M);
    int fe;
    float fm = frexpf(F, &fe);
    int s = fe - 1;
    float x = 2.0f * fm;
    float L = oz2o_log2f(x);
    float lg = f32_add_dir(L, (float)s, FE_UPWARD);          /* eq. (7) */
    float prod = f32_mul_dir(c->delta, lg, FE_UPWARD);
    float d = f32_sub_dir(c->Paccu, prod, FE_DOWNWARD);
    return (5 - E) + (int)floorf(d);
}

/* abar = ceil(|a| 2^(5-E)) in [0, 64] */
static int ceil_scaled_abs(double a, int E)
{
    if (a == 0.0) return 0;
    uint64_t M; int q;
    decompose(a, &M, &q);
    long sh = (long)q + 5 - E;              /* value = M 2^sh, < 64 */
    if (sh >= 0) return (int)(M << sh);     /* cannot exceed 64; only when M small: never for M >= 2^52 */
    if (-sh >= 64) return 1;
    uint64_t fl = M >> (-sh);
    uint64_t rem = M & ((((uint64_t)1) << (-sh)) - 1);
    return (int)fl + (rem != 0);
}

/* ------------------------------------------------------------------------------------ */
/* O2 + O3: exponents e[m] (rows of A) and f[n] (columns of B); mu_i = 2^e_i, nu_j = 2^f_j */
/* Optional outputs (may be NULL): EA[m], EB[n] = floor(log2 max); SA[m], SB[n] = Sfix;   */
/* rowmax[m], colmax[n] = max_j cbar_ij, max_i cbar_ij (accurate mode only).             */
/* mode: 0 accurate, 1 original fast (Alg.1), 2 revised fast (Alg.2).                    */
/* ------------------------------------------------------------------------------------ */
int oz2o_exponents(int mode, int N, long m, long n, long k,
                   const double *A, long lda, const double *B, long ldb,
                   int32_t *e, int32_t *f, int32_t *EA, int32_t *EB,
                   uint64_t *SA, uint64_t *SB, int64_t *rowmax, int64_t *colmax)
{
    oz_consts c;
    if (oz_make_consts(N, &c)) return -1;
    if (mode < 0 || mode > 2) return -2;
    int32_t *Ea = malloc(sizeof(int32_t) * (size_t)(m > 0 ? m : 1));
    int32_t *Eb = malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
    uint64_t *Sa = malloc(sizeof(uint64_t) * (size_t)(m > 0 ? m : 1));
    uint64_t *Sb = malloc(sizeof(uint64_t) * (size_t)(n > 0 ? n : 1));
    char *nzA = malloc((size_t)(m > 0 ? m : 1)), *nzB = malloc((size_t)(n > 0 ? n : 1));
#pragma omp parallel for schedule(static)
    for (long i = 0; i < m; i++) {
        int E; uint64_t S;
        nzA[i] = (char)(vec_stats(A + i, (size_t)lda, k, &E, &S) > 0);
        Ea[i] = E; Sa[i] = S;
    }
#pragma omp parallel for schedule(static)
    for (long j = 0; j < n; j++) {
        int E; uint64_t S;
        nzB[j] = (char)(vec_stats(B + (size_t)j * (size_t)ldb, 1, k, &E, &S) > 0);
        Eb[j] = E; Sb[j] = S;
    }
    if (mode == 1 || mode == 2) {
        for (long i = 0; i < m; i++) e[i] = nzA[i] ? exponent_fast_or_prop(mode, &c, Ea[i], Sa[i], sq_shift(k)) : 0;
        for (long j = 0; j < n; j++) f[j] = nzB[j] ? exponent_fast_or_prop(mode, &c, Eb[j], Sb[j], sq_shift(k)) : 0;
    } else {
        /* accurate mode: Abar, Bbar, Cbar = Abar Bbar, row/col maxima */
        int8_t *Ab = malloc((size_t)m * (size_t)k + 1), *Bb = malloc((size_t)k * (size_t)n + 1);
        int64_t *rmx = calloc((size_t)(m > 0 ? m : 1), sizeof(int64_t));
        int64_t *cmx = calloc((size_t)(n > 0 ? n : 1), sizeof(int64_t));
#pragma omp parallel for schedule(static)
        for (long i = 0; i < m; i++)
            for (long h = 0; h < k; h++)
                Ab[(size_t)i * k + h] = (int8_t)(nzA[i] ? ceil_scaled_abs(CM(A, lda, i, h), Ea[i]) : 0);
#pragma omp parallel for schedule(static)
        for (long j = 0; j < n; j++)
            for (long h = 0; h < k; h++)
                Bb[(size_t)j * k + h] = (int8_t)(nzB[j] ? ceil_scaled_abs(CM(B, ldb, h, j), Eb[j]) : 0);
#pragma omp parallel
        {
            int64_t *cloc = calloc((size_t)(n > 0 ? n : 1), sizeof(int64_t));
#pragma omp for schedule(static)
            for (long i = 0; i < m; i++) {
                const int8_t *ar = Ab + (size_t)i * k;
                int64_t rm = 0;
                for (long j = 0; j < n; j++) {
                    const int8_t *bc = Bb + (size_t)j * k;
                    int64_t s = 0;
                    for (long h = 0; h < k; h++) s += (int32_t)ar[h] * (int32_t)bc[h];
                    if (s > rm) rm = s;
                    if (s > cloc[j]) cloc[j] = s;
                }
                rmx[i] = rm;
            }
#pragma omp critical
            for (long j = 0; j < n; j++)
                if (cloc[j] > cmx[j]) cmx[j] = cloc[j];
            free(cloc);
        }
        for (long i = 0; i < m; i++) e[i] = nzA[i] ? exponent_accurate(&c, Ea[i], rmx[i]) : 0;
        for (long j = 0; j < n; j++) f[j] = nzB[j] ? exponent_accurate(&c, Eb[j], cmx[j]) : 0;
        if (rowmax) memcpy(rowmax, rmx, sizeof(int64_t) * (size_t)m);
        if (colmax) memcpy(colmax, cmx, sizeof(int64_t) * (size_t)n);
        free(Ab); free(Bb); free(rmx); free(cmx);
    }
    if (EA) memcpy(EA, Ea, sizeof(int32_t) * (size_t)m);
    if (EB) memcpy(EB, Eb, sizeof(int32_t) * (size_t)n);
    if (SA) memcpy(SA, Sa, sizeof(uint64_t) * (size_t)m);
    if (SB) memcpy(SB, Sb, sizeof(uint64_t) * (size_t)n);
    free(Ea); free(Eb); free(Sa); free(Sb); free(nzA); free(nzB);
    return 0;
}

/* ------------------------------------------------------------------------------------ */
/* O4: a' = trunc(a * 2^e) exactly (Step 2).  Returns 1 if |a'| >= 2^126.       */
/* ------------------------------------------------------------------------------------ */
static int trunc_scaled(double a, int e, i128 *out)
{
    if (a == 0.0) { *out = 0; return 0; }
    uint64_t M; int q;
    decompose(a, &M, &q);
    long sh = (long)q + e;
    u128 V;
    if (sh >= 0) {
        if (sh > 73) { *out = 0; return 1; }    /* 53 + 73 = 126 bits */
        V = (u128)M << sh;
    } else if (-sh >= 64) V = 0;
    else V = (u128)(M >> (-sh));                /* dropping bits of the magnitude = toward zero */
    *out = (a < 0) ? -(i128)V : (i128)V;
    return 0;
}

/* A' as pairs (lo, hi) of 64-bit words of the two's-complement 128-bit value; layout:
 * op == 0: rows of A, out[(i*k + h)*2 ..];  op == 1: columns of B, out[(j*k + h)*2 ..].   */
int oz2o_truncate(int op, long rows, long k, const double *X, long ldx, const int32_t *ex, uint64_t *out)
{
    int bad = 0;
#pragma omp parallel for schedule(static) reduction(| : bad)
    for (long r = 0; r < rows; r++)
        for (long h = 0; h < k; h++) {
            double a = op == 0 ? CM(X, ldx, r, h) : CM(X, ldx, h, r);
            i128 v;
            bad |= trunc_scaled(a, ex[r], &v);
            out[((size_t)r * k + h) * 2 + 0] = (uint64_t)(u128)v;
            out[((size_t)r * k + h) * 2 + 1] = (uint64_t)((u128)v >> 64);
        }
    return bad ? -3 : 0;
}

/* ------------------------------------------------------------------------------------ */
/* O5: symmetric INT8 residue of a' modulo p (reading R5)                   */
/* ------------------------------------------------------------------------------------ */
static int8_t sym_residue(i128 v, int p)
{
    int u = (int)(v % p);                   /* C remainder: sign of v */
    if (u < 0) u += p;                      /* u = v mod p in [0, p) */
    if (u > (p - 1) / 2) u -= p;            /* symmetric representative; p = 256 -> [-128, 127] */
    return (int8_t)u;
}

/* residues of op(X) scaled by ex: out[l][r][h], r over rows of A (op 0) / columns of B (op 1) */
int oz2o_residues(int op, int N, long rows, long k, const double *X, long ldx, const int32_t *ex, int8_t *out)
{
    oz_consts c;
    if (oz_make_consts(N, &c)) return -1;
    int bad = 0;
#pragma omp parallel for schedule(static) reduction(| : bad)
    for (long r = 0; r < rows; r++)
        for (long h = 0; h < k; h++) {
            double a = op == 0 ? CM(X, ldx, r, h) : CM(X, ldx, h, r);
            i128 v;
            bad |= trunc_scaled(a, ex[r], &v);
            for (int l = 0; l < N; l++)
                out[((size_t)l * rows + r) * k + h] = sym_residue(v, c.p[l]);
        }
    return bad ? -3 : 0;
}

/* ------------------------------------------------------------------------------------ */
/* O6: U_l[j][i] = (sum_h rA_l[i][h] rB_l[j][h]) mod p_l in [0,p_l)  (eq. (2));    */
/* maxabs_R = max |sum| over everything (INT32 headroom).                         */
/* ------------------------------------------------------------------------------------ */
int oz2o_products(int N, long m, long n, long k, const int8_t *RA, const int8_t *RB, uint8_t *U, int64_t *maxabs_R)
{
    oz_consts c;
    if (oz_make_consts(N, &c)) return -1;
    int64_t mx = 0;
    for (int l = 0; l < N; l++) {
        const int8_t *ra = RA + (size_t)l * m * k, *rb = RB + (size_t)l * n * k;
        int p = c.p[l];
#pragma omp parallel for schedule(static) reduction(max : mx)
        for (long j = 0; j < n; j++)
            for (long i = 0; i < m; i++) {
                const int8_t *x = ra + (size_t)i * k, *y = rb + (size_t)j * k;
                int64_t s = 0;
                for (long h = 0; h < k; h++) s += (int32_t)x[h] * (int32_t)y[h];
                int64_t a = s < 0 ? -s : s;
                if (a > mx) mx = a;
                int64_t u = s % p;
                if (u < 0) u += p;
                U[((size_t)l * n + j) * m + i] = (uint8_t)u;
            }
    }
    if (maxabs_R) *maxabs_R = mx;
    return 0;
}

/* ------------------------------------------------------------------------------------ */
/* O7: C' = sum_l w_l U_l ; C'' = rmod(C', P) in [-P/2, P/2)  (eq. (2)(3); reading R7)   */
/* ------------------------------------------------------------------------------------ */
static wint crt_combine(const oz_consts *c, const uint8_t *u /* N residues */)
{
    wint acc = w_zero();
    for (int l = 0; l < c->N; l++) acc = w_add(acc, w_mul_u64(c->w[l], (uint64_t)u[l]));
    /* 0 <= acc < N * 256 * P < 2^13 P : subtract P 2^b, b = 13..0 */
    for (int b = 13; b >= 0; b--) {
        wint t = w_shl(c->P, b);
        if (w_cmp(acc, t) >= 0) acc = w_sub(acc, t);
    }
    /* acc in [0, P); symmetric: acc - P if 2 acc >= P */
    if (w_cmp(w_shl(acc, 1), c->P) >= 0) acc = w_sub(acc, c->P);
    return acc;
}

/* Cpp: [n][m][4] u64 words (two's complement, little-endian), m fastest */
int oz2o_crt(int N, long m, long n, const uint8_t *U, uint64_t *Cpp)
{
    oz_consts c;
    if (oz_make_consts(N, &c)) return -1;
#pragma omp parallel for schedule(static)
    for (long j = 0; j < n; j++)
        for (long i = 0; i < m; i++) {
            uint8_t u[OZ_MAX_MODULI];
            for (int l = 0; l < N; l++) u[l] = U[((size_t)l * n + j) * m + i];
            wint r = crt_combine(&c, u);
            memcpy(Cpp + ((size_t)j * m + i) * 4, r.w, 32);
        }
    return 0;
}

/* ------------------------------------------------------------------------------------ */
/* O8: exact Z = A'B' and Zabs = sum |a'||b'| in 256-bit integers; condition (1).   */
/* Ap: [m][k] (lo,hi) pairs, Bp: [n][k] pairs (from oz2o_truncate).                      */
/* Z, Zabs: [n][m][4] words (may be NULL).  counts[0] = #{2 Zabs >= P} (condition (1)     */
/* violated), counts[1] = #{Z outside [-P/2, P/2)} (recovery actually wrong).            */
/* ------------------------------------------------------------------------------------ */
static i128 load_i128(const uint64_t *p) { return (i128)(((u128)p[1] << 64) | p[0]); }

int oz2o_exact_product(int N, long m, long n, long k, const uint64_t *Ap, const uint64_t *Bp,
                       uint64_t *Z, uint64_t *Zabs, int64_t *counts)
{
    oz_consts c;
    if (oz_make_consts(N, &c)) return -1;
    int64_t viol = 0, wrong = 0;
    wint negP = w_neg(c.P);
#pragma omp parallel for schedule(static) reduction(+ : viol, wrong)
    for (long j = 0; j < n; j++)
        for (long i = 0; i < m; i++) {
            wint z = w_zero(), za = w_zero();
            for (long h = 0; h < k; h++) {
                i128 a = load_i128(Ap + ((size_t)i * k + h) * 2);
                i128 b = load_i128(Bp + ((size_t)j * k + h) * 2);
                wint pr = w_mul_i128(a, b);
                z = w_add(z, pr);
                za = w_add(za, w_abs(pr));
            }
            if (w_cmp(w_shl(za, 1), c.P) >= 0) viol++;
            wint z2 = w_shl(z, 1);                      /* |z| < 2^254 guaranteed by widths */
            if (!(w_cmp(z2, c.P) < 0 && w_cmp(z2, negP) >= 0)) wrong++;
            if (Z) memcpy(Z + ((size_t)j * m + i) * 4, z.w, 32);
            if (Zabs) memcpy(Zabs + ((size_t)j * m + i) * 4, za.w, 32);
        }
    if (counts) { counts[0] = viol; counts[1] = wrong; }
    return 0;
}

/* ------------------------------------------------------------------------------------ */
/* O9: C = RN_64(C'') 2^-(e_i+f_j) ; out = alpha C (+ beta C_in)  (Step 4; R8, R9)        */
/* ------------------------------------------------------------------------------------ */
int oz2o_unscale(long m, long n, const uint64_t *Cpp, const int32_t *e, const int32_t *f,
                 double alpha, double beta, double *C, long ldc)
{
#pragma omp parallel for schedule(static)
    for (long j = 0; j < n; j++)
        for (long i = 0; i < m; i++) {
            wint v;
            memcpy(v.w, Cpp + ((size_t)j * m + i) * 4, 32);
            double cij = w_to_double_scaled(v, -((long)e[i] + (long)f[j]));
            double t = alpha * cij;
            double *dst = &CM(C, ldc, i, j);
            *dst = (beta == 0.0) ? t : fma(beta, *dst, t);
        }
    return 0;
}

/* RN_64(v 2^sh) of a 256-bit word vector, for the tests */
double oz2o_words_to_double(const uint64_t *words, long sh)
{
    wint v;
    memcpy(v.w, words, 32);
    return w_to_double_scaled(v, sh);
}

/* ------------------------------------------------------------------------------------ */
/* The whole path in one call (Steps 1-4), used for timing the oracle and as the          */
/* end-to-end reference.  Returns 0, or a negative code.  Optional outputs may be NULL.   */
/* ------------------------------------------------------------------------------------ */
int oz2o_dgemm(long m, long n, long k, double alpha, const double *A, long lda,
               const double *B, long ldb, double beta, double *C, long ldc,
               int N, int mode, int32_t *e_out, int32_t *f_out)
{
    if (m < 0 || n < 0 || k < 0) return -1;
    if (m == 0 || n == 0) return 0;
    int rc = 0;
    int32_t *e = malloc(sizeof(int32_t) * (size_t)m), *f = malloc(sizeof(int32_t) * (size_t)n);
    size_t ka = (size_t)(k > 0 ? k : 1);
    int8_t *RA = malloc((size_t)N * m * ka), *RB = malloc((size_t)N * n * ka);
    uint8_t *U = malloc((size_t)N * m * n);
    uint64_t *Cpp = malloc((size_t)m * n * 32);
    if (!e || !f || !RA || !RB || !U || !Cpp) { rc = -9; goto done; }
    rc = oz2o_exponents(mode, N, m, n, k, A, lda, B, ldb, e, f, 0, 0, 0, 0, 0, 0);
    if (rc) goto done;
    rc = oz2o_residues(0, N, m, k, A, lda, e, RA);
    if (rc) goto done;
    rc = oz2o_residues(1, N, n, k, B, ldb, f, RB);
    if (rc) goto done;
    rc = oz2o_products(N, m, n, k, RA, RB, U, 0);
    if (rc) goto done;
    rc = oz2o_crt(N, m, n, U, Cpp);
    if (rc) goto done;
    rc = oz2o_unscale(m, n, Cpp, e, f, alpha, beta, C, ldc);
    if (e_out) memcpy(e_out, e, sizeof(int32_t) * (size_t)m);
    if (f_out) memcpy(f_out, f, sizeof(int32_t) * (size_t)n);
done:
    free(e); free(f); free(RA); free(RB); free(U); free(Cpp);
    return rc;
}

/* ------------------------------------------------------------------------------------ */
/* SGEMM variant (Fig. 6): FP32 in, FP32 out.  Every float is a double, */
/* so Steps 1-3 are the FP64 path on the promoted inputs (the scaling formulas do not       */
/* depend on the input precision); only Step 4 changes:               */
/*   c = RN_32(C'' 2^-(e_i+f_j))  -- one rounding of the exact integer to FP32 --           */
/*   out = alpha c (+ beta C_in) in FP32  (readings R8, R9 with FP32 in place of FP64).     */
/* ------------------------------------------------------------------------------------ */
static float w_to_float_scaled(wint v, long sh)
{
    if (w_iszero(v)) return 0.0f;
    int neg = w_isneg(v);
    wint a = w_abs(v);
    int t = w_bitlen(a) - 1;               /* a in [2^t, 2^(t+1)) */
    long E = (long)t + sh;                 /* value in [2^E, 2^(E+1)) */
    long qe = E - 23;                      /* exponent of the last kept bit (24-bit significand) */
    if (qe < -149) qe = -149;              /* FP32 subnormal quantum */
    long r = qe - sh;                      /* bits of a dropped below the quantum */
    uint64_t q;
    if (r <= 0) {
        q = a.w[0] << (-r);                /* nothing dropped: a has at most 24 bits here */
    } else if (r > 256) {
        q = 0;
    } else {
        q = 0;
        for (int b = 0; b < 25; b++) q |= (uint64_t)w_bit(a, (int)r + b) << b;
        int half = w_bit(a, (int)r - 1);
        int sticky = 0;
        for (int b = 0; b < (int)r - 1 && !sticky; b++) sticky = w_bit(a, b);
        if (half && (sticky || (q & 1))) q += 1;
    }
    float d = ldexpf((float)q, (int)qe);   /* q <= 2^24: exact; overflows to inf */
    return neg ? -d : d;
}

float oz2o_words_to_float(const uint64_t *words, long sh)
{
    wint v;
    memcpy(v.w, words, 32);
    return w_to_float_scaled(v, sh);
}

int oz2o_unscale_f32(long m, long n, const uint64_t *Cpp, const int32_t *e, const int32_t *f,
                     float alpha, float beta, float *C, long ldc)
{
#pragma omp parallel for schedule(static)
    for (long j = 0; j < n; j++)
        for (long i = 0; i < m; i++) {
            wint v;
            memcpy(v.w, Cpp + ((size_t)j * m + i) * 4, 32);
            float cij = w_to_float_scaled(v, -((long)e[i] + (long)f[j]));
            volatile float t = alpha * cij;
            float *dst = &C[(size_t)j * ldc + i];
            *dst = (beta == 0.0f) ? t : fmaf(beta, *dst, t);
        }
    return 0;
}

int oz2o_sgemm(long m, long n, long k, float alpha, const float *A, long lda,
               const float *B, long ldb, float beta, float *C, long ldc,
               int N, int mode, int32_t *e_out, int32_t *f_out)
{
    if (m < 0 || n < 0 || k < 0) return -1;
    if (m == 0 || n == 0) return 0;
    int rc = 0;
    size_t ka = (size_t)(k > 0 ? k : 1);
    double *Ad = malloc(sizeof(double) * (size_t)m * ka), *Bd = malloc(sizeof(double) * ka * (size_t)n);
    int32_t *e = malloc(sizeof(int32_t) * (size_t)m), *f = malloc(sizeof(int32_t) * (size_t)n);
    int8_t *RA = malloc((size_t)N * m * ka), *RB = malloc((size_t)N * n * ka);
    uint8_t *U = malloc((size_t)N * m * n);
    uint64_t *Cpp = malloc((size_t)m * n * 32);
    if (!Ad || !Bd || !e || !f || !RA || !RB || !U || !Cpp) { rc = -9; goto done; }
    for (long h = 0; h < k; h++)
        for (long i = 0; i < m; i++) Ad[(size_t)h * m + i] = (double)A[(size_t)h * lda + i];       /* exact */
    for (long j = 0; j < n; j++)
        for (long h = 0; h < k; h++) Bd[(size_t)j * k + h] = (double)B[(size_t)j * ldb + h];
    long ldad = m > 1 ? m : 1, ldbd = k > 1 ? k : 1;
    rc = oz2o_exponents(mode, N, m, n, k, Ad, ldad, Bd, ldbd, e, f, 0, 0, 0, 0, 0, 0);
    if (rc) goto done;
    rc = oz2o_residues(0, N, m, k, Ad, ldad, e, RA);
    if (rc) goto done;
    rc = oz2o_residues(1, N, n, k, Bd, ldbd, f, RB);
    if (rc) goto done;
    rc = oz2o_products(N, m, n, k, RA, RB, U, 0);
    if (rc) goto done;
    rc = oz2o_crt(N, m, n, U, Cpp);
    if (rc) goto done;
    rc = oz2o_unscale_f32(m, n, Cpp, e, f, alpha, beta, C, ldc);
    if (e_out) memcpy(e_out, e, sizeof(int32_t) * (size_t)m);
    if (f_out) memcpy(f_out, f, sizeof(int32_t) * (size_t)n);
done:
    free(Ad); free(Bd); free(e); free(f); free(RA); free(RB); free(U); free(Cpp);
    return rc;
}

/* ------------------------------------------------------------------------------------ */
/* O10: reference AB in double-double: two-product by fma, two-sum accumulation.  */
/* hi, lo: [n][m] column-major contiguous (ld = m).                                       */
/* ------------------------------------------------------------------------------------ */
int oz2o_dd_reference(long m, long n, long k, const double *A, long lda, const double *B, long ldb,
                      double *hi, double *lo)
{
#pragma omp parallel for schedule(static)
    for (long j = 0; j < n; j++)
        for (long i = 0; i < m; i++) {
            double sh = 0.0, sl = 0.0;
            for (long h = 0; h < k; h++) {
                double a = CM(A, lda, i, h), b = CM(B, ldb, h, j);
                double p = a * b;
                double pe = fma(a, b, -p);              /* p + pe = a b exactly */
                double s = sh + p;                      /* two-sum */
                double bb = s - sh;
                double se = (sh - (s - bb)) + (p - bb);
                se += sl + pe;
                sh = s + se;                            /* fast two-sum renormalisation */
                sl = se - (sh - s);
            }
            hi[(size_t)j * m + i] = sh;
            lo[(size_t)j * m + i] = sl;
        }
    return 0;
}

int oz2o_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
