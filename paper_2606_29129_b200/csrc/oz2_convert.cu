// oz2_convert.cu -- S2: A' = trunc(diag(mu) A), B' = trunc(B diag(nu)) (Step 2) and the symmetric
// INT8 residues rmod(., p_l) for all N moduli in ONE pass over A and B.
//
// Arithmetic.  |a'| (up to 84 bits, never written to memory) lives in registers as NB 32-bit words.  With d_i the
// base-256 digits of |a'|, for an odd modulus p
//     x = sum_i d_i (256^i mod p)                                       (NB dp4a; x < 2^20, congruent to |a'|)
// and the symmetric residue is r = sign(a') (x - p round(x / p)).  The reduction runs in FP32 on exact small
// integers, so that it can use both halves of the FMA pipe (integer multiplies only run on one):
//     the dp4a chain starts from 0x4B000000, the bit pattern of 2^23, so its result read as a float is 2^23 + x;
//     q = RN(x (1/p)~ + 1.5 2^23) - 1.5 2^23 is round(x / p) exactly: |x (1/p)~ - x/p| < 2^-11, while x / p is at
//     least 1/(2p) > 2^-9 away from every half-integer (p odd);
//     x - q p is then exact, and RN(sign (x - q p) + 1.5 2^23) holds r in two's complement in its low byte.
// p = 256: the low byte of a' in two's complement (reading R5).
//
// Data movement (the stage is bound by HBM traffic 8 + N bytes per element and by ~7 integer instructions per
// element and modulus).  Planes are [l][row][kp], k fastest (K-major for the tensor-core GEMM),
// kp = round_up(k, 128), zero padded.  Work unit everywhere: a "quad" = 4 consecutive h of one row, held by one
// lane, so that a warp stores 128 contiguous bytes per row and modulus.
//   * B is column-major = already K-major: a warp streams 256 consecutive h of one column with 16-byte loads.
//   * A is column-major = M-major: a CTA stages a 32-row x 128-h tile through shared memory (coalesced 256-byte
//     reads along the rows, transposed on the way in), then every warp converts whole rows of the tile.
// The same two movers serve accurate mode's Abar / Bbar = ceil(mu' |.|), one plane.
#include "oz2_common.cuh"

namespace {

struct ConvTab {
    float invp, negp;          // RN(1 / p), -p
    uint32_t wb[3];            // byte weights 256^(4t+b) mod p, packed
    uint32_t pad[3];
};
__constant__ ConvTab c_conv[OZ2_MAX_MODULI];

constexpr int TI = 32;             // rows of A per tile
constexpr int TH = 128;            // h per tile
constexpr int SROW = TH + 2;       // padded row of the staging tile in doubles (16-byte aligned rows)
constexpr int CONV_THREADS = 256;

// magnitude words of trunc(|a| 2^ex); returns the sign mask of a (0 or 0xFFFFFFFF)
template <int NB>
__device__ __forceinline__ uint32_t scaled_words(double a, int ex, uint32_t (&w)[NB])
{
    const unsigned long long b = (unsigned long long)__double_as_longlong(a);
    const uint32_t hi = (uint32_t)(b >> 32), lo = (uint32_t)b;
    const uint32_t negm = (uint32_t)((int32_t)hi >> 31);
    const int be = (int)((hi >> 20) & 0x7FFu);
    const uint32_t m1 = (hi & 0x000FFFFFu) | (be ? 0x00100000u : 0u), m0 = lo;
    const unsigned long long M = ((unsigned long long)m1 << 32) | m0;
    const int sh = (be ? be : 1) - 1075 + ex;          // |a| 2^ex = M 2^sh, M < 2^53
    if (NB == 2) {
        // |a'| < 2^64: a non-zero M is shifted left by at most 63
        unsigned long long v;
        if (sh >= 0) v = M << (sh > 63 ? 63 : sh);
        else v = (-sh < 64) ? (M >> (-sh)) : 0ull;      // dropping magnitude bits = toward zero
        w[0] = (uint32_t)v;
        w[1] = (uint32_t)(v >> 32);
    } else {
        if (sh >= 0) {
            // |a'| < 2^96: word shift ws = sh / 32 (<= 2 for a non-zero M), bit shift bs
            const int s = sh > 95 ? 95 : sh;
            const int ws = s >> 5, bs = s & 31;
            const uint32_t t0 = m0 << bs, t1 = __funnelshift_l(m0, m1, bs), t2 = __funnelshift_l(m1, 0u, bs);
            w[0] = ws == 0 ? t0 : 0u;
            w[1] = ws == 0 ? t1 : (ws == 1 ? t0 : 0u);
            w[2] = ws == 0 ? t2 : (ws == 1 ? t1 : t0);
        } else {
            const int r = -sh;
            const unsigned long long v = r < 64 ? (M >> r) : 0ull;
            w[0] = (uint32_t)v;
            w[1] = (uint32_t)(v >> 32);
            w[2] = 0u;
        }
    }
    return negm;
}

// Two quads at once (8 elements, exponents ex0 / ex1): residues for every modulus, one 4-byte store per quad and
// modulus.  The per-modulus constants are loaded once for the 8 elements; `ok1` guards the second quad's stores.
template <int NB>
__device__ __forceinline__ void oct_residues(const double (&a)[2][4], int ex0, int ex1, int N, int8_t *dst0,
                                             int64_t dst1_off, bool ok1, int64_t plane_stride)
{
    constexpr float MAGIC = 12582912.0f;               // 1.5 2^23: RN(y + MAGIC) - MAGIC = round(y) for |y| < 2^22
    uint32_t w[8][NB];
    float sg[8];                                       // +1.0f / -1.0f
    uint32_t b256[8];                                  // a' in two's complement, low word
#pragma unroll
    for (int u = 0; u < 8; u++) {
        const uint32_t negm = scaled_words<NB>(a[u >> 2][u & 3], u < 4 ? ex0 : ex1, w[u]);
        sg[u] = __uint_as_float(0x3F800000u | (negm & 0x80000000u));
        b256[u] = (w[u][0] ^ negm) - negm;
    }
    int8_t *out = dst0;
    {   // p = 256: low bytes
        const uint32_t lo = __byte_perm(b256[0], b256[1], 0x0040), hi = __byte_perm(b256[2], b256[3], 0x0040);
        *reinterpret_cast<uint32_t *>(out) = __byte_perm(lo, hi, 0x5410);
        const uint32_t lo1 = __byte_perm(b256[4], b256[5], 0x0040), hi1 = __byte_perm(b256[6], b256[7], 0x0040);
        if (ok1) *reinterpret_cast<uint32_t *>(out + dst1_off) = __byte_perm(lo1, hi1, 0x5410);
    }
#pragma unroll 1
    for (int l = 1; l < N; l++) {
        const float invp = c_conv[l].invp, negp = c_conv[l].negp;
        const uint32_t wb0 = c_conv[l].wb[0], wb1 = c_conv[l].wb[1], wb2 = c_conv[l].wb[2];
        uint32_t r[8];
#pragma unroll
        for (int u = 0; u < 8; u++) {
            uint32_t xb = __dp4a(w[u][0], wb0, 0x4B000000u);
            xb = __dp4a(w[u][1], wb1, xb);
            if (NB == 3) xb = __dp4a(w[u][2], wb2, xb);
            const float x = __fadd_rn(__uint_as_float(xb), -8388608.0f);        // exact
            const float q = __fadd_rn(__fmaf_rn(x, invp, MAGIC), -MAGIC);       // round(x / p), exact
            const float rm = __fmaf_rn(q, negp, x);                             // x - q p in [-(p-1)/2, (p-1)/2]
            r[u] = __float_as_uint(__fmaf_rn(rm, sg[u], MAGIC));                // low byte = sign * rm
        }
        out += plane_stride;
        const uint32_t lo = __byte_perm(r[0], r[1], 0x0040), hi = __byte_perm(r[2], r[3], 0x0040);
        *reinterpret_cast<uint32_t *>(out) = __byte_perm(lo, hi, 0x5410);
        const uint32_t lo1 = __byte_perm(r[4], r[5], 0x0040), hi1 = __byte_perm(r[6], r[7], 0x0040);
        if (ok1) *reinterpret_cast<uint32_t *>(out + dst1_off) = __byte_perm(lo1, hi1, 0x5410);
    }
}

// accurate mode: ceil(|a| 2^(5-E)) in [0, 64]
__device__ __forceinline__ uint32_t ceil_scaled(double a, int E)
{
    const unsigned long long b = (unsigned long long)__double_as_longlong(a) & 0x7FFFFFFFFFFFFFFFull;
    if (b == 0) return 0u;
    const int be = (int)(b >> 52);
    const unsigned long long mant = b & 0x000FFFFFFFFFFFFFull;
    const unsigned long long M = be ? (mant | 0x0010000000000000ull) : mant;
    const int q = (be ? be : 1) - 1075;
    const int r = -(q + 5 - E);           // value = M 2^-r <= 64; r >= 47 for normal numbers
    if (r <= 0) return (uint32_t)(M << (-r));
    if (r >= 64) return 1u;
    return (uint32_t)(M >> r) + ((M & ((1ull << r) - 1)) != 0 ? 1u : 0u);
}

__device__ __forceinline__ void quad_bar(const double (&a)[4], int E, int8_t *dst)
{
    uint32_t o = 0;
#pragma unroll
    for (int u = 0; u < 4; u++) o |= ceil_scaled(a[u], E) << (8 * u);
    *reinterpret_cast<uint32_t *>(dst) = o;
}

// ---------------------------------------------------------------------------------------------
// A path.  MODE 0: residues (NB words)   MODE 1: Abar
// ---------------------------------------------------------------------------------------------
template <int NB, int MODE, typename T>
__global__ void __launch_bounds__(CONV_THREADS)
k2_rows(int N, int64_t m, int64_t k, const T *__restrict__ A, int64_t lda, const int32_t *__restrict__ e,
        int8_t *__restrict__ planes, int64_t kp)
{
    __shared__ __align__(16) double tile[TI * SROW];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t i0 = (int64_t)blockIdx.x * TI, h0 = (int64_t)blockIdx.y * TH;
    // ---- stage: thread (lane = row, warp = h mod 8), 16 loads in flight, transposed into tile[i][h]
    {
        const int64_t i = i0 + lane;
        const bool iok = i < m;
        const T *src = A + i + (h0 + warp) * lda;
        double v[16];
#pragma unroll
        for (int s = 0; s < 16; s++) {
            const int64_t h = h0 + warp + 8 * s;
            v[s] = (iok && h < k) ? (double)__ldg(src + (int64_t)(8 * s) * lda) : 0.0;
        }
#pragma unroll
        for (int s = 0; s < 16; s++) tile[lane * SROW + warp + 8 * s] = v[s];
    }
    __syncthreads();
    // ---- convert: warp w owns rows 4w .. 4w+3, lane owns the quad h = 4 lane .. 4 lane + 3
    const int64_t plane_stride = m * kp;
#pragma unroll 1
    for (int rr = 0; rr < TI / 8; rr += 2) {
        const int il = warp * (TI / 8) + rr;
        const int64_t i = i0 + il;
        if (i >= m) break;
        const bool ok1 = i + 1 < m;
        double a[2][4];
#pragma unroll
        for (int t = 0; t < 2; t++) {
            const double2 lo = *reinterpret_cast<const double2 *>(&tile[(il + t) * SROW + 4 * lane]);
            const double2 hi = *reinterpret_cast<const double2 *>(&tile[(il + t) * SROW + 4 * lane + 2]);
            a[t][0] = lo.x; a[t][1] = lo.y; a[t][2] = hi.x; a[t][3] = hi.y;
        }
        int8_t *dst = planes + i * kp + h0 + 4 * lane;
        const int ex0 = __ldg(e + i), ex1 = ok1 ? __ldg(e + i + 1) : 0;
        if (MODE == 0) oct_residues<NB>(a, ex0, ex1, N, dst, kp, ok1, plane_stride);
        else {
            quad_bar(a[0], ex0, dst);
            if (ok1) quad_bar(a[1], ex1, dst + kp);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// B path: warp = 256 consecutive h of column j; lane holds the quads at 4 lane and 128 + 4 lane
// ---------------------------------------------------------------------------------------------
// four consecutive elements of a column as doubles: two 16-byte loads (FP64) or one (FP32)
__device__ __forceinline__ void ld4(const double *p, double (&a)[4])
{
    const double2 v0 = __ldg(reinterpret_cast<const double2 *>(p)), v1 = __ldg(reinterpret_cast<const double2 *>(p + 2));
    a[0] = v0.x; a[1] = v0.y; a[2] = v1.x; a[3] = v1.y;
}
__device__ __forceinline__ void ld4(const float *p, double (&a)[4])
{
    const float4 v = __ldg(reinterpret_cast<const float4 *>(p));
    a[0] = (double)v.x; a[1] = (double)v.y; a[2] = (double)v.z; a[3] = (double)v.w;
}

template <int NB, int MODE, typename T>
__global__ void __launch_bounds__(CONV_THREADS)
k2_cols(int N, int64_t n, int64_t k, const T *__restrict__ B, int64_t ldb, const int32_t *__restrict__ f,
        int8_t *__restrict__ planes, int64_t kp)
{
    const int lane = threadIdx.x & 31;
    const int64_t chunks = (kp + 255) / 256;
    const int64_t item = (int64_t)blockIdx.x * (CONV_THREADS / 32) + (threadIdx.x >> 5);
    if (item >= n * chunks) return;
    const int64_t j = item / chunks, c = item - j * chunks;
    const T *col = B + j * ldb;
    const int ex = __ldg(f + j);
    const bool vec = ((((uintptr_t)col) & 15) == 0);
    const int64_t plane_stride = n * kp;
    double a[2][4];
#pragma unroll
    for (int t = 0; t < 2; t++) {
        const int64_t h = c * 256 + 128 * t + 4 * lane;
        if (vec && h + 3 < k) {
            ld4(col + h, a[t]);
        } else {
#pragma unroll
            for (int u = 0; u < 4; u++) a[t][u] = (h + u < k) ? (double)__ldg(col + h + u) : 0.0;
        }
    }
    const int64_t h = c * 256 + 4 * lane;           // first quad; kp is a multiple of 128, so it is inside
    int8_t *dst = planes + j * kp + h;
    const bool ok1 = h + 128 < kp;
    if (MODE == 0) oct_residues<NB>(a, ex, ex, N, dst, 128, ok1, plane_stride);
    else {
        quad_bar(a[0], ex, dst);
        if (ok1) quad_bar(a[1], ex, dst + 128);
    }
}

} // namespace

int oz2_convert_upload_tables(const Oz2HostTables &t)
{
    ConvTab h[OZ2_MAX_MODULI];
    for (int l = 0; l < OZ2_MAX_MODULI; l++) {
        const uint32_t p = t.mod[l].p;
        h[l].invp = (float)(1.0 / (double)p);
        h[l].negp = -(float)p;
        for (int i = 0; i < 3; i++) { h[l].wb[i] = t.mod[l].wb[i]; h[l].pad[i] = 0; }
    }
    OZ2_CUDA_TRY(cudaMemcpyToSymbol(c_conv, h, sizeof(h)));
    return 0;
}

template <typename T>
static int launch_convert_t(int op, int N, int wide, int64_t rows, int64_t k, const T *X, int64_t ldx, const int32_t *ex,
                            int8_t *planes, int64_t kp, cudaStream_t st)
{
    if (op == 0) {
        dim3 grid((unsigned)((rows + TI - 1) / TI), (unsigned)(kp / TH));
        if (N == 0) k2_rows<2, 1, T><<<grid, CONV_THREADS, 0, st>>>(N, rows, k, X, ldx, ex, planes, kp);
        else if (wide) k2_rows<3, 0, T><<<grid, CONV_THREADS, 0, st>>>(N, rows, k, X, ldx, ex, planes, kp);
        else k2_rows<2, 0, T><<<grid, CONV_THREADS, 0, st>>>(N, rows, k, X, ldx, ex, planes, kp);
    } else {
        const int64_t items = rows * ((kp + 255) / 256);
        const unsigned gx = (unsigned)((items + CONV_THREADS / 32 - 1) / (CONV_THREADS / 32));
        if (N == 0) k2_cols<2, 1, T><<<gx, CONV_THREADS, 0, st>>>(N, rows, k, X, ldx, ex, planes, kp);
        else if (wide) k2_cols<3, 0, T><<<gx, CONV_THREADS, 0, st>>>(N, rows, k, X, ldx, ex, planes, kp);
        else k2_cols<2, 0, T><<<gx, CONV_THREADS, 0, st>>>(N, rows, k, X, ldx, ex, planes, kp);
    }
    oz2_count_launches(1);
    OZ2_CUDA_TRY(cudaGetLastError());
    return 0;
}

// op 0: rows of A, op 1: columns of B.  N >= 1: residue planes [N][rows][kp] with exponents `ex`.  N == 0: the
// single plane ceil(mu' |.|) of accurate mode; `ex` then holds E = floor(log2 max |.|) per row.
// f32 != 0: X is FP32 (SGEMM variant), promoted exactly on load.
int oz2_launch_convert(int op, int N, int wide, int f32, int64_t rows, int64_t k, const void *X, int64_t ldx,
                       const int32_t *ex, int8_t *planes, int64_t kp, cudaStream_t st)
{
    if (rows <= 0) return 0;
    if (f32) return launch_convert_t<float>(op, N, wide, rows, k, static_cast<const float *>(X), ldx, ex, planes, kp, st);
    return launch_convert_t<double>(op, N, wide, rows, k, static_cast<const double *>(X), ldx, ex, planes, kp, st);
}
