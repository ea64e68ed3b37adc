// oz2_scale.cu -- S1: the scaling vectors mu_i = 2^e_i (rows of A), nu_j = 2^f_j (columns of B).
//
//   mode 2  revised fast mode, Algorithm 2, eq. (17)(18)
//   mode 1  original fast mode, Algorithm 1, eq. (11)(12)
//   mode 0  accurate mode, eq. (4)-(9): max exponents, Abar/Bbar = ceil(mu'|a|);
//           the auxiliary INT8 GEMM itself runs in oz2_gemm.cu with a row/column-max epilogue.
//
// Readings: R2 the sum of squares is the exact integer sum_h ceil(2^44 (v_h / 2^E)^2) -- order
// independent, so it can be accumulated with integer atomics; R3 __log2f is replaced by the correctly
// rounded RN_32(log2 x); R10/R11 directed roundings and the normalised form of Algorithm 2.
//
// Kernels are HBM-bound streaming reductions: A is column-major, so a warp reads 32 consecutive rows of one
// column (coalesced) and every thread keeps the statistics of its own row; a column of B is contiguous and is
// reduced by one block with warp shuffles.
#include "oz2_common.cuh"

#include <mutex>

namespace {

__constant__ Oz2CrtTab c_crt[OZ2_MAX_MODULI + 1];

constexpr int ROWS_PER_BLOCK = 128;   // consecutive rows of A per block (1 KB contiguous per column)
constexpr int KSLICES = 2;            // h-interleaved slices inside a block
constexpr int COL_THREADS = 256;
constexpr int32_t OZ2_E_ZERO = INT32_MIN;   // marks an all-zero row / column in the E arrays of accurate mode

__device__ __forceinline__ unsigned long long abs_bits(double v)
{
    return (unsigned long long)__double_as_longlong(v) & 0x7FFFFFFFFFFFFFFFull;
}

// floor(log2 v) for the positive finite double with bit pattern `b` (true value for subnormals)
__device__ __forceinline__ int floor_log2_bits(unsigned long long b)
{
    int be = (int)(b >> 52);
    if (be) return be - 1023;
    return (63 - __clzll((long long)b)) - 1074;
}

// |v| = M 2^q, M < 2^53 integer
__device__ __forceinline__ void decompose(unsigned long long b, unsigned long long &M, int &q)
{
    int be = (int)(b >> 52);
    unsigned long long mant = b & 0x000FFFFFFFFFFFFFull;
    M = be ? (mant | 0x0010000000000000ull) : mant;
    q = (be ? be : 1) - 1075;
}

// T = ceil(2^44 (v / 2^E)^2) for |v| < 2^(E+1): exact.  (reading R2)
// Slow path, any input: exact 128-bit integer square.
__device__ __noinline__ unsigned long long sq_term_int(unsigned long long b, int E, int SQ)
{
    unsigned long long M;
    int q;
    decompose(b, M, q);
    // 2^SQ (v/2^E)^2 = M^2 2^-s with s = 2 (E - q) - SQ.
    int s = 2 * (E - q) - SQ;
    unsigned long long lo = M * M, hi = __umul64hi(M, M);
    if (s <= 0) return lo << (-s);                    // exact, the value is at most 2^46
    if (s < 64) return ((hi << (64 - s)) | (lo >> s)) + ((lo & ((1ull << s) - 1)) ? 1ull : 0ull);
    if (s < 128) {
        int r = s - 64;
        unsigned long long rem = (r ? (hi & ((1ull << r) - 1)) : 0ull) | lo;
        return (hi >> r) + (rem ? 1ull : 0ull);
    }
    return 1ull;
}

// Fast path: x = |v| 2^(22-E) is an exact exponent shift while it stays a normal number (x < 2^23), x^2 < 2^46 has
// a quantum <= 2^-7 in FP64, so RU(x x) <= ceil(x^2) (integers below 2^53 are representable) and
// ceil(RU(x x)) = ceil(x^2) exactly: one DMUL.RU and one F2I.CEIL.
// SQ (even; 44 for k <= 2^17, reading R2b beyond) is the fixed-point position of the sum.
__device__ __forceinline__ unsigned long long sq_term(unsigned long long b, int E, int SQ)
{
    if (b == 0) return 0;
    const int be = (int)(b >> 52);
    const int hs = (SQ >> 1) - E;                     // x = |v| 2^hs
    const int ne = be + hs;                           // biased exponent of x
    if (be == 0 || ne < 1) return sq_term_int(b, E, SQ);  // subnormal input or subnormal x: rare
    const double x = __longlong_as_double((long long)(b + ((unsigned long long)(long long)hs << 52)));
    return __double2ull_ru(__dmul_ru(x, x));
}

// The same term for a whole vector whose E is known: x = RU(|v| 2^hs) with the scale 2^hs, hs = SQ/2 - E, held as a double.
// While x is a normal number the product is an exact exponent shift; when it underflows, rounding up keeps 0 < x < 1, so
// that ceil(RU(x x)) = 1 = ceil(x^2) as it must; v = 0 gives 0.  Three FP64 instructions per element instead of the
// exponent-field arithmetic of sq_term.  Needs 2^hs representable: sq_scale_ok(E, SQ).
__device__ __forceinline__ bool sq_scale_ok(int E, int SQ) { const int hs = (SQ >> 1) - E; return hs >= -1022 && hs <= 1023; }
__device__ __forceinline__ double sq_scale(int E, int SQ) { return __longlong_as_double((long long)((SQ >> 1) - E + 1023) << 52); }
__device__ __forceinline__ unsigned long long sq_term_scaled(double v, double scale)
{
    const double x = __dmul_ru(fabs(v), scale);
    return __double2ull_ru(__dmul_ru(x, x));
}

// max |v| over a vector is needed only through floor(log2 .) and "is it zero": for normal numbers the high word of the
// bit pattern decides both, so the streaming loops keep a 32-bit maximum of the high words (sign bit cleared); only a
// vector whose high-word maximum stays below 2^20 (nothing but subnormals and zeros) is re-read for the exact pattern.
__device__ __forceinline__ uint32_t hi_abs(double v) { return (uint32_t)__double2hiint(v) & 0x7FFFFFFFu; }
constexpr uint32_t HI_NORMAL = 0x00100000u;

// LOG2F(x) = RN_32(log2 x) for float x in [1,2] (reading R3): FP64 log2 (<= 1 ulp), rounded once.
__device__ __forceinline__ float log2f_rn(float x) { return __double2float_rn(log2((double)x)); }

// Algorithm 2 (mode 2) / Algorithm 1 (mode 1) on the statistics (E, S) of one row or column.
__device__ int exponent_fastprop(int mode, const Oz2CrtTab &c, unsigned long long amax, unsigned long long S, int SQ)
{
    if (amax == 0) return 0;                                            // reading R4
    int E = floor_log2_bits(amax);
    float F = __ull2float_ru(S);                                        // "rounding-up"
    int fb = __float_as_int(F);
    int shat = ((fb >> 23) - 127) - SQ;                                 // floor(log2 F) - SQ
    float x = __int_as_float((fb & 0x007FFFFF) | 0x3F800000);           // F / 2^floor(log2 F) in [1,2)
    float L = log2f_rn(x);
    if (mode == 2) {
        float t = __fmaf_ru(0.5f, L, 1.1920928955078125e-07f);          // single_up(0.5 __log2f(.) + 2 u32)
        float w = __fsub_rd(c.Pprop, 0.5f * (float)shat);               // single_down(P'_prop - 0.5 s)
        float d = __fsub_rd(w, t);
        return (int)floorf(d) - E;
    } else {
        int s = shat + 2 * E;                                           // floor(log2 a_norm), raw sum
        float inner = __fadd_ru(L, (float)s);
        float t = __fmul_ru(c.delta, inner);                            // single_up(delta (__log2f(.) + s))
        float d = __fsub_rd(c.Pfast, fmaxf(t, 1.0f));
        return (int)floorf(d) - E;
    }
}

// eq. (8)/(9) with reading G3: e = (5 - E) + floor(P'_accu - delta log2~(max cbar)); log2~ of eq. (7)
__device__ int exponent_accurate(const Oz2CrtTab &c, int E, int M)
{
    if (M < 1) M = 1;
    float F = __uint2float_ru((unsigned)M);
    int fb = __float_as_int(F);
    int s = (fb >> 23) - 127;
    float x = __int_as_float((fb & 0x007FFFFF) | 0x3F800000);
    float L = log2f_rn(x);
    float lg = __fadd_ru(L, (float)s);
    float prod = __fmul_ru(c.delta, lg);
    float d = __fsub_rd(c.Pprop, prod);
    return (5 - E) + (int)floorf(d);
}

// ---------------------------------------------------------------------------------------------
// rows of A
// ---------------------------------------------------------------------------------------------
template <int PASS, typename T> // PASS 0: max |a|   1: sum of squared, normalised terms;  T: double or float (SGEMM)
__global__ void __launch_bounds__(ROWS_PER_BLOCK *KSLICES)
k1_rows(int64_t m, int64_t k, const T *__restrict__ A, int64_t lda, int64_t kchunk,
        unsigned long long *__restrict__ amax, unsigned long long *__restrict__ ssq, int SQ)
{
    pdl_launch_dependents();
    pdl_wait();                                  // PASS 1 reads the maxima of PASS 0; every kernel of the chain waits (transitivity)
    int64_t i = (int64_t)blockIdx.x * ROWS_PER_BLOCK + threadIdx.x;
    int64_t h0 = (int64_t)blockIdx.y * kchunk;
    int64_t h1 = h0 + kchunk < k ? h0 + kchunk : k;
    if (i >= m) return;
    const T *p = A + i;
    if (PASS == 0) {
        uint32_t mh = 0;
        int64_t h = h0 + threadIdx.y;
        for (; h + 7 * KSLICES < h1; h += 8 * KSLICES) {
            double v[8];
#pragma unroll
            for (int u = 0; u < 8; u++) v[u] = (double)__ldg(p + (h + u * KSLICES) * lda);
#pragma unroll
            for (int u = 0; u < 8; u++) mh = max(mh, hi_abs(v[u]));
        }
        for (; h < h1; h += KSLICES) mh = max(mh, hi_abs((double)__ldg(p + h * lda)));
        if (mh >= HI_NORMAL) {
            atomicMax(amax + i, (unsigned long long)mh << 32);    // same floor(log2 .) as the exact pattern
        } else {
            // nothing but subnormals and zeros in this slice (rare): exact 64-bit pattern
            unsigned long long acc = 0;
            for (int64_t hh = h0 + threadIdx.y; hh < h1; hh += KSLICES) {
                const unsigned long long b = abs_bits((double)__ldg(p + hh * lda));
                acc = b > acc ? b : acc;
            }
            if (acc) atomicMax(amax + i, acc);
        }
    } else {
        const unsigned long long mx = amax[i];
        if (mx == 0) return;
        const int E = floor_log2_bits(mx);
        unsigned long long acc = 0;
        int64_t h = h0 + threadIdx.y;
        if (sq_scale_ok(E, SQ)) {
            const double scale = sq_scale(E, SQ);
            for (; h + 7 * KSLICES < h1; h += 8 * KSLICES) {
                double v[8];
#pragma unroll
                for (int u = 0; u < 8; u++) v[u] = (double)__ldg(p + (h + u * KSLICES) * lda);
#pragma unroll
                for (int u = 0; u < 8; u++) acc += sq_term_scaled(v[u], scale);
            }
            for (; h < h1; h += KSLICES) acc += sq_term_scaled((double)__ldg(p + h * lda), scale);
        } else {
            for (; h < h1; h += KSLICES) acc += sq_term(abs_bits((double)__ldg(p + h * lda)), E, SQ);
        }
        if (acc) atomicAdd(ssq + i, acc);
    }
}

__global__ void k1_rows_finalize(int mode, int N, int64_t m, const unsigned long long *__restrict__ amax,
                                 const unsigned long long *__restrict__ ssq, int32_t *__restrict__ e, int SQ)
{
    pdl_launch_dependents();
    pdl_wait();
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < m) e[i] = exponent_fastprop(mode, c_crt[N], amax[i], ssq[i], SQ);
}

// ---------------------------------------------------------------------------------------------
// columns of B: one block per column
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long block_reduce(unsigned long long v, bool is_max, unsigned long long *sm)
{
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        unsigned long long w = __shfl_xor_sync(0xffffffffu, v, o);
        v = is_max ? (w > v ? w : v) : v + w;
    }
    int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();
    if (lane == 0) sm[warp] = v;
    __syncthreads();
    unsigned long long r = sm[0];
    for (int w = 1; w < COL_THREADS / 32; w++) r = is_max ? (sm[w] > r ? sm[w] : r) : r + sm[w];
    return r;
}

// MODE 1/2: f[j]; MODE 0 (accurate prepare): EB[j] only
// two consecutive elements of a column as doubles (16-byte load for FP64, 8-byte for FP32)
__device__ __forceinline__ double2 ld2(const double *p) { return __ldg(reinterpret_cast<const double2 *>(p)); }
__device__ __forceinline__ double2 ld2(const float *p)
{
    const float2 v = __ldg(reinterpret_cast<const float2 *>(p));
    return make_double2((double)v.x, (double)v.y);
}

template <bool ACCU, typename T>
__global__ void __launch_bounds__(COL_THREADS)
k1_cols(int mode, int N, int64_t k, const T *__restrict__ B, int64_t ldb, int32_t *__restrict__ f,
        int32_t *__restrict__ EB, int SQ)
{
    __shared__ unsigned long long sm[COL_THREADS / 32];
    pdl_launch_dependents();
    pdl_wait();
    const T *col = B + (int64_t)blockIdx.x * ldb;
    bool vec = ((((uintptr_t)col) & (2 * sizeof(T) - 1)) == 0);
    int64_t kv = vec ? (k & ~(int64_t)1) : 0;
    uint32_t mh = 0;
    for (int64_t h = 2 * (int64_t)threadIdx.x; h < kv; h += 2 * COL_THREADS) {
        double2 v = ld2(col + h);
        mh = max(mh, max(hi_abs(v.x), hi_abs(v.y)));
    }
    for (int64_t h = kv + threadIdx.x; h < k; h += COL_THREADS) mh = max(mh, hi_abs((double)__ldg(col + h)));
    unsigned long long mx = block_reduce((unsigned long long)mh << 32, true, sm);
    if (mx < ((unsigned long long)HI_NORMAL << 32)) {
        // nothing but subnormals and zeros in this column (rare; uniform for the block): exact 64-bit pattern
        unsigned long long acc = 0;
        for (int64_t h = threadIdx.x; h < k; h += COL_THREADS) {
            const unsigned long long b = abs_bits((double)__ldg(col + h));
            acc = b > acc ? b : acc;
        }
        mx = block_reduce(acc, true, sm);
    }
    if (ACCU) {
        if (threadIdx.x == 0) EB[blockIdx.x] = mx ? floor_log2_bits(mx) : OZ2_E_ZERO;
        return;
    }
    if (mx == 0) {
        if (threadIdx.x == 0) f[blockIdx.x] = 0;
        return;
    }
    int E = floor_log2_bits(mx);
    unsigned long long acc = 0;
    if (sq_scale_ok(E, SQ)) {                                                           // uniform for the block
        const double scale = sq_scale(E, SQ);
        for (int64_t h = 2 * (int64_t)threadIdx.x; h < kv; h += 2 * COL_THREADS) {      // second read: L2 hits
            double2 v = ld2(col + h);
            acc += sq_term_scaled(v.x, scale) + sq_term_scaled(v.y, scale);
        }
        for (int64_t h = kv + threadIdx.x; h < k; h += COL_THREADS) acc += sq_term_scaled((double)__ldg(col + h), scale);
    } else {
        for (int64_t h = threadIdx.x; h < k; h += COL_THREADS) acc += sq_term(abs_bits((double)__ldg(col + h)), E, SQ);
    }
    acc = block_reduce(acc, false, sm);
    if (threadIdx.x == 0) f[blockIdx.x] = exponent_fastprop(mode, c_crt[N], mx, acc, SQ);
}

// ---------------------------------------------------------------------------------------------
// accurate mode: E per row / column; Abar, Bbar are written by the movers of oz2_convert.cu
// ---------------------------------------------------------------------------------------------
__global__ void k1_rows_E(int64_t m, const unsigned long long *__restrict__ amax, int32_t *__restrict__ EA)
{
    pdl_launch_dependents();
    pdl_wait();
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < m) EA[i] = amax[i] ? floor_log2_bits(amax[i]) : OZ2_E_ZERO;
}

__global__ void k1_accu_finalize(int N, int64_t cnt, const int32_t *__restrict__ E, const int32_t *__restrict__ mx,
                                 int32_t *__restrict__ out)
{
    pdl_launch_dependents();
    pdl_wait();
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= cnt) return;
    // a zero row / column (E == OZ2_E_ZERO) gets exponent 0 (reading R4)
    out[i] = E[i] == OZ2_E_ZERO ? 0 : exponent_accurate(c_crt[N], E[i], mx[i]);
}

__global__ void k_log2f(const float *__restrict__ x, float *__restrict__ y, int64_t count)
{
    int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t < count) y[t] = log2f_rn(x[t]);
}

// fixed-point position of the rounded-up sum of squares (reading R2 / R2b)
int sq_shift(int64_t k)
{
    int lg = 0;
    while (((int64_t)1 << lg) < k) lg++;
    const int extra = lg > 17 ? lg - 17 : 0;
    return 44 - 2 * ((extra + 1) / 2);
}

int rows_grid_y(int64_t m, int64_t k, int64_t *kchunk)
{
    int64_t bx = (m + ROWS_PER_BLOCK - 1) / ROWS_PER_BLOCK;
    int64_t want = (148 * 8 + bx - 1) / bx;               // >= 8 blocks per SM overall
    int64_t maxy = (k + 16 * KSLICES - 1) / (16 * KSLICES);
    if (want > maxy) want = maxy;
    if (want < 1) want = 1;
    if (want > 65535) want = 65535;
    int64_t kc = (k + want - 1) / want;
    kc = oz2_round_up(kc, 8 * KSLICES);
    *kchunk = kc;
    return (int)((k + kc - 1) / kc);
}

} // namespace

int oz2_scale_upload_tables(const Oz2HostTables &t)
{
    OZ2_CUDA_TRY(cudaMemcpyToSymbol(c_crt, t.crt, sizeof(t.crt)));
    return 0;
}

int oz2_launch_scale_rows(int mode, int N, int f32, int64_t m, int64_t k, const void *Av, int64_t lda,
                          unsigned long long *amaxA, unsigned long long *ssqA, int32_t *e, cudaStream_t st)
{
    const double *A = static_cast<const double *>(Av);
    const float *Af = static_cast<const float *>(Av);
    if (m <= 0) return 0;
    // the two statistics arrays are neighbours in the workspace: one memset node instead of two when they are
    const char *lo = reinterpret_cast<const char *>(amaxA), *hi = reinterpret_cast<const char *>(ssqA + m);
    if (ssqA > amaxA && (size_t)(hi - lo) <= 16 * (size_t)m + 1024) {
        OZ2_CUDA_TRY(cudaMemsetAsync(amaxA, 0, (size_t)(hi - lo), st));
    } else {
        OZ2_CUDA_TRY(cudaMemsetAsync(amaxA, 0, sizeof(unsigned long long) * (size_t)m, st));
        OZ2_CUDA_TRY(cudaMemsetAsync(ssqA, 0, sizeof(unsigned long long) * (size_t)m, st));
    }
    int64_t kchunk;
    int gy = rows_grid_y(m, k, &kchunk);
    dim3 grid((unsigned)((m + ROWS_PER_BLOCK - 1) / ROWS_PER_BLOCK), (unsigned)gy), block(ROWS_PER_BLOCK, KSLICES);
    if (f32) {
        OZ2_CUDA_TRY(oz2_launch(k1_rows<0, float>, grid, block, 0, st, m, k, Af, lda, kchunk, amaxA, ssqA, sq_shift(k)));
        OZ2_CUDA_TRY(oz2_launch(k1_rows<1, float>, grid, block, 0, st, m, k, Af, lda, kchunk, amaxA, ssqA, sq_shift(k)));
    } else {
        OZ2_CUDA_TRY(oz2_launch(k1_rows<0, double>, grid, block, 0, st, m, k, A, lda, kchunk, amaxA, ssqA, sq_shift(k)));
        OZ2_CUDA_TRY(oz2_launch(k1_rows<1, double>, grid, block, 0, st, m, k, A, lda, kchunk, amaxA, ssqA, sq_shift(k)));
    }
    OZ2_CUDA_TRY(oz2_launch(k1_rows_finalize, dim3((unsigned)((m + 255) / 256)), dim3(256), 0, st, mode, N, m, amaxA, ssqA, e, sq_shift(k)));
    oz2_count_launches(3);
    OZ2_CUDA_TRY(cudaGetLastError());
    return 0;
}

int oz2_launch_scale_cols(int mode, int N, int f32, int64_t n, int64_t k, const void *B, int64_t ldb, int32_t *f, cudaStream_t st)
{
    if (n <= 0) return 0;
    if (f32) OZ2_CUDA_TRY(oz2_launch(k1_cols<false, float>, dim3((unsigned)n), dim3(COL_THREADS), 0, st, mode, N, k, static_cast<const float *>(B), ldb, f, nullptr, sq_shift(k)));
    else OZ2_CUDA_TRY(oz2_launch(k1_cols<false, double>, dim3((unsigned)n), dim3(COL_THREADS), 0, st, mode, N, k, static_cast<const double *>(B), ldb, f, nullptr, sq_shift(k)));
    oz2_count_launches(1);
    OZ2_CUDA_TRY(cudaGetLastError());
    return 0;
}

// accurate mode, one side: E[i] = floor(log2 max_h |x_ih|) for the `cnt` vectors of length k of X, and the INT8 plane
// ceil(|x| 2^(5-E)).  strided != 0: vector i is X[i + h ldx] (rows of a column-major matrix), else
// X[h + i ldx] (its columns).  amax: u64 scratch of `cnt` entries (strided side only).
int oz2_launch_scale_accu_side(int f32, int strided, int64_t cnt, int64_t k, const void *X, int64_t ldx,
                               unsigned long long *amax, int32_t *E, int8_t *bar, int64_t kp, cudaStream_t st)
{
    if (cnt <= 0) return 0;
    if (strided) {
        OZ2_CUDA_TRY(cudaMemsetAsync(amax, 0, sizeof(unsigned long long) * (size_t)cnt, st));
        int64_t kchunk;
        int gy = rows_grid_y(cnt, k, &kchunk);
        dim3 grid((unsigned)((cnt + ROWS_PER_BLOCK - 1) / ROWS_PER_BLOCK), (unsigned)gy), block(ROWS_PER_BLOCK, KSLICES);
        if (f32) OZ2_CUDA_TRY(oz2_launch(k1_rows<0, float>, grid, block, 0, st, cnt, k, static_cast<const float *>(X), ldx, kchunk, amax, (unsigned long long *)nullptr, 44));
        else OZ2_CUDA_TRY(oz2_launch(k1_rows<0, double>, grid, block, 0, st, cnt, k, static_cast<const double *>(X), ldx, kchunk, amax, (unsigned long long *)nullptr, 44));
        OZ2_CUDA_TRY(oz2_launch(k1_rows_E, dim3((unsigned)((cnt + 255) / 256)), dim3(256), 0, st, cnt, amax, E));
        oz2_count_launches(2);
    } else {
        if (f32) OZ2_CUDA_TRY(oz2_launch(k1_cols<true, float>, dim3((unsigned)cnt), dim3(COL_THREADS), 0, st, 0, 2, k, static_cast<const float *>(X), ldx, (int32_t *)nullptr, E, 44));
        else OZ2_CUDA_TRY(oz2_launch(k1_cols<true, double>, dim3((unsigned)cnt), dim3(COL_THREADS), 0, st, 0, 2, k, static_cast<const double *>(X), ldx, (int32_t *)nullptr, E, 44));
        oz2_count_launches(1);
    }
    OZ2_CUDA_TRY(cudaGetLastError());
    return oz2_launch_convert(strided ? 0 : 1, 0, 0, f32, cnt, k, X, ldx, E, bar, kp, st);
}

int oz2_launch_scale_accu_finish(int N, int64_t m, int64_t n, const int32_t *EA, const int32_t *EB,
                                 const int32_t *rowmax, const int32_t *colmax, int32_t *e, int32_t *f, cudaStream_t st)
{
    OZ2_CUDA_TRY(oz2_launch(k1_accu_finalize, dim3((unsigned)((m + 255) / 256)), dim3(256), 0, st, N, m, EA, rowmax, e));
    OZ2_CUDA_TRY(oz2_launch(k1_accu_finalize, dim3((unsigned)((n + 255) / 256)), dim3(256), 0, st, N, n, EB, colmax, f));
    oz2_count_launches(2);
    OZ2_CUDA_TRY(cudaGetLastError());
    return 0;
}

int oz2_launch_log2f(const float *x, float *y, int64_t count, cudaStream_t st)
{
    if (count <= 0) return 0;
    k_log2f<<<(unsigned)((count + 255) / 256), 256, 0, st>>>(x, y, count);
    oz2_count_launches(1);
    OZ2_CUDA_TRY(cudaGetLastError());
    return 0;
}

// ---------------------------------------------------------------------------------------------
// ozaki2_row_exponents_noalloc: the row kernels above with their statistics in memory the library brings along
// ---------------------------------------------------------------------------------------------
// For callers that cannot hand us a workspace because they cannot allocate one: a plug-in whose host application
// owns all device memory, a control loop that must not stall the device in cudaMalloc, a component that may not touch
// the driver's allocator after start-up.  k1_rows<0> / k1_rows<1> / k1_rows_finalize need 16 bytes of scratch per
// row (amax[i], ssq[i]); here those come from a fixed array in the module's data segment: 2 x 65536 x 8 B = 1 MiB,
// loaded with the library on every GPU that uses it and released only at process exit.
//
// The identifier below means two different things.  Inside a kernel it is the array.  In host code it is only the
// handle the runtime registered for it -- not a device address -- so it must never be passed to a kernel or to
// cudaMemsetAsync as it stands: the device address is asked for with cudaGetSymbolAddress, once per device (each
// device has its own copy at its own address) while that device is current, and that address is what the kernels get.
namespace {

static __device__ __align__(256) unsigned long long g_noalloc_row_stats[2 * OZ2_NOALLOC_MAX_ROWS];

constexpr int NOALLOC_MAX_DEVICES = 64;
unsigned long long *g_noalloc_addr[NOALLOC_MAX_DEVICES];   // device address of g_noalloc_row_stats, per device; null = not asked yet
std::mutex g_noalloc_mu;

// Set-up on first use per device.  No allocation: the array already exists on the device.
int noalloc_row_stats(unsigned long long **out)
{
    int dev = -1;
    OZ2_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return (int)cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lk(g_noalloc_mu);
    if (!g_noalloc_addr[dev]) {
        void *p = nullptr;
        const cudaError_t rc = cudaGetSymbolAddress(&p, g_noalloc_row_stats);    // address on the CURRENT device
        if (rc != cudaSuccess) return (int)rc;
        if (!p || (reinterpret_cast<uintptr_t>(p) & 255)) return (int)cudaErrorInvalidSymbol;
        g_noalloc_addr[dev] = static_cast<unsigned long long *>(p);
    }
    *out = g_noalloc_addr[dev];
    return 0;
}

} // namespace

int oz2_launch_scale_rows_noalloc(int mode, int N, int64_t m, int64_t k, const double *A, int64_t lda, int32_t *e, cudaStream_t st)
{
    if (m <= 0) return 0;
    if (m > OZ2_NOALLOC_MAX_ROWS) return (int)cudaErrorInvalidValue;           // the entry point has refused this already
    unsigned long long *stats = nullptr;
    const int rc = noalloc_row_stats(&stats);
    if (rc) return rc;
    // amax[0..m) and ssq[0..m) side by side (256-byte aligned), so that the launcher zeroes exactly the 16 m bytes this
    // call uses with one stream-ordered memset: the array still holds the statistics of whichever call ran before
    unsigned long long *amax = stats, *ssq = stats + oz2_round_up(m, 32);
    return oz2_launch_scale_rows(mode, N, 0, m, k, A, lda, amax, ssq, e, st);
}
