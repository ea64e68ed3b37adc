// oz2_crt.cu -- S4 + S5: CRT reconstruction and unscaling.
//
//   C'  = sum_l w_l U_l,  w_l = P_l q_l                       (eq. (2); Theorem 1)
//   C'' = rmod(C', P) in [-P/2, P/2)                           (eq. (3); reading R7)
//   C   = RN_64(C'') 2^-(e_i+f_j)                              (Step 4; reading R8)
//   out = alpha C (+ beta C_in)                                (reading R9)
//
// Everything up to the single rounding RN_64 is EXACT integer arithmetic on 32-bit words held in registers
// (the weights have up to 156 bits, C' up to 169): sum_l w_{l,t} U_l per word with 64-bit accumulators,
// carry propagation, a quotient estimate Q ~ C'/P in FP64 (|error| < 2^-30; the rare near-half cases take an
// exact compare against P/2), C'' = C' - Q P, then a 64-bit normalised mantissa with a sticky bit is rounded
// once.  HBM traffic: N bytes in + 8 bytes out per element; the kernel is templated on N so that all weight
// words are constant-bank operands of fully unrolled multiply-adds.
#include "oz2_common.cuh"

namespace {

__constant__ Oz2CrtTab c_crt[OZ2_MAX_MODULI + 1];

// number of 32-bit words of P for N moduli (log2 P: 15.99, 23.98, 31.95, 39.9, ... 155.4)
__host__ __device__ constexpr int words_of_P(int N)
{
    return N <= 4 ? 1 : N <= 8 ? 2 : N <= 12 ? 3 : N <= 16 ? 4 : 5;
}

// RN of (mant64 | sticky) * 2^sc with a single rounding, subnormals and overflow included
__device__ __noinline__ double round_scaled_slow(unsigned long long mant, uint32_t sticky, int sc)
{
    // value in [2^(63+sc), 2^(64+sc))
    int Ex = 63 + sc;
    if (Ex > 1023) return __longlong_as_double(0x7FF0000000000000ll);
    int rs = -1074 - sc;                          // bits dropped below the subnormal quantum 2^-1074
    if (rs < 11) rs = 11;                         // never keep more than 53 bits
    unsigned long long q, half, low;
    if (rs >= 65) return 0.0;
    if (rs == 64) { q = 0; half = mant >> 63; low = (mant << 1) | sticky; }
    else { q = mant >> rs; half = (mant >> (rs - 1)) & 1ull; low = (mant & ((1ull << (rs - 1)) - 1)) | sticky; }
    if (half && (low || (q & 1ull))) q += 1;
    // q * 2^(sc + rs)
    int qe = sc + rs;
    if (qe == -1074) return __longlong_as_double((long long)q);       // subnormal (or the smallest normal)
    double d = (double)(long long)q;                                   // q <= 2^53: exact
    // qe > -1074 here means the result is normal; scale in two exact steps to stay in range
    int h1 = qe / 2, h2 = qe - h1;
    d *= __longlong_as_double((long long)(h1 + 1023) << 52);
    d *= __longlong_as_double((long long)(h2 + 1023) << 52);
    return d;
}

template <int N>
__device__ __forceinline__ double crt_one(const uint32_t (&u)[N], int esum, uint64_t *cpp_out)
{
    constexpr int NW = words_of_P(N);
    const Oz2CrtTab &T = c_crt[N];
    // ---- C' = sum_l w_l U_l, word by word
    unsigned long long acc[NW];
#pragma unroll
    for (int t = 0; t < NW; t++) acc[t] = 0;
#pragma unroll
    for (int l = 0; l < N; l++)
#pragma unroll
        for (int t = 0; t < NW; t++) acc[t] += (unsigned long long)T.w[l][t] * u[l];
    uint32_t c[NW + 1];
    unsigned long long carry = 0;
#pragma unroll
    for (int t = 0; t < NW; t++) {
        unsigned long long s = acc[t] + carry;
        c[t] = (uint32_t)s;
        carry = s >> 32;
    }
    c[NW] = (uint32_t)carry;                                          // < 2^13
    // ---- Q = round(C' / P), estimated from the top three words
    double top = (double)(long long)(((unsigned long long)c[NW] << 32) | c[NW - 1]);
    if constexpr (NW >= 2) top = fma((double)c[NW - 2], 2.3283064365386963e-10, top);
    double qd = top * T.invP;                                         // invP holds 2^(32 (NW-1)) / P
    double qr = floor(qd + 0.5);
    uint32_t Q = (uint32_t)(int)qr;
    bool near_half = fabs(qd - qr) > 0.5 - 9.5367431640625e-07;       // 2^-20 guard, estimate error < 2^-30
    // ---- R = C' - Q P (two's complement, NW + 1 words)
    uint32_t r[NW + 1];
    long long br = 0;
#pragma unroll
    for (int t = 0; t <= NW; t++) {
        long long s = (long long)c[t] + br - (long long)((unsigned long long)Q * (t < NW ? T.P[t] : 0u));
        r[t] = (uint32_t)s;
        br = s >> 32;
    }
    if (near_half) {
        // exact: bring R into [-P/2, P/2)
        for (int pass = 0; pass < 2; pass++) {
            bool neg = (r[NW] >> 31) != 0;
            // d = R - P/2 (if R >= 0) or R + P/2 (if R < 0)
            uint32_t d[NW + 1];
            long long b2 = 0;
            for (int t = 0; t <= NW; t++) {
                long long ph = t < NW ? (long long)T.Phalf[t] : 0ll;
                long long s = (long long)r[t] + b2 + (neg ? ph : -ph);
                d[t] = (uint32_t)s;
                b2 = s >> 32;
            }
            bool dneg = (d[NW] >> 31) != 0;
            bool fix = neg ? dneg : !dneg;        // R < -P/2  or  R >= P/2
            if (!fix) break;
            long long b3 = 0;
            for (int t = 0; t <= NW; t++) {
                long long pw = t < NW ? (long long)T.P[t] : 0ll;
                long long s = (long long)r[t] + b3 + (neg ? pw : -pw);
                r[t] = (uint32_t)s;
                b3 = s >> 32;
            }
        }
    }
    const uint32_t negm = (uint32_t)((int32_t)r[NW] >> 31);
    if (cpp_out) {
        uint32_t w8[8];
#pragma unroll
        for (int t = 0; t < 8; t++) w8[t] = t <= NW ? r[t] : negm;
#pragma unroll
        for (int t = 0; t < 4; t++) cpp_out[t] = ((unsigned long long)w8[2 * t + 1] << 32) | w8[2 * t];
    }
    // ---- |C''| as three 64-bit pieces X2:X1:X0 (|C''| <= P/2 < 2^(32 NW) <= 2^160), branch-free negate
    const unsigned long long m64 = (unsigned long long)(long long)(int32_t)negm;
    auto W = [&](int t) -> uint32_t { return t <= NW ? r[t <= NW ? t : 0] : negm; };   // sign-extended word t
    const unsigned long long R0 = ((unsigned long long)W(1) << 32) | W(0);
    const unsigned long long R1 = ((unsigned long long)W(3) << 32) | W(2);
    const unsigned long long R2 = ((unsigned long long)W(5) << 32) | W(4);
    // two's-complement negate of the 192-bit value when negative: X = (R ^ m) + (m & 1)
    const unsigned long long X0 = (R0 ^ m64) + (m64 & 1ull);
    const unsigned long long c0 = (m64 & 1ull) & (unsigned long long)(X0 == 0ull);
    const unsigned long long X1 = (R1 ^ m64) + c0;
    const unsigned long long c1 = c0 & (unsigned long long)(X1 == 0ull);
    const unsigned long long X2 = (R2 ^ m64) + c1;
    // ---- leading piece, top 64 bits from the leading one, sticky bit
    unsigned long long ptop, pmid, plow;
    int base;
    if (NW >= 5 && X2 != 0ull) { ptop = X2; pmid = X1; plow = X0; base = 128; }
    else if (NW >= 3 && X1 != 0ull) { ptop = X1; pmid = X0; plow = 0ull; base = 64; }
    else { ptop = X0; pmid = 0ull; plow = 0ull; base = 0; }
    if (ptop == 0ull) return 0.0;
    const int lz = __clzll((long long)ptop);
    const unsigned long long mant = (ptop << lz) | ((pmid >> 1) >> (63 - lz));
    const uint32_t sticky = (((pmid << lz) | plow) != 0ull) ? 1u : 0u;
    const int pos = base + 63 - lz;                                   // |C''| in [2^pos, 2^(pos+1))
    const int sc = pos - 63 - esum;                                   // result = mant 2^sc
    double v;
    const int Ex = pos - esum;
    if (Ex >= -1020 && Ex <= 1021) {
        const double d = __ull2double_rn(mant | sticky);              // the one rounding, ties to even
        v = __longlong_as_double(__double_as_longlong(d) + ((long long)sc << 52));
    } else {
        v = round_scaled_slow(mant, sticky, sc);
    }
    return __longlong_as_double(__double_as_longlong(v) | (long long)(m64 << 63));
}

template <int N, bool WANT_CPP>
__global__ void __launch_bounds__(128)
k4_crt(int64_t m, int64_t n, const uint8_t *__restrict__ U, int64_t mp, const int32_t *__restrict__ e,
       const int32_t *__restrict__ f, double alpha, double beta, double *__restrict__ C, int64_t ldc,
       uint64_t *__restrict__ Cpp)
{
    const int64_t i0 = 4 * ((int64_t)blockIdx.y * 128 + threadIdx.x);
    const int64_t j = blockIdx.x;
    if (i0 >= m) return;
    const int64_t plane = n * mp;
    uint32_t packed[N];
#pragma unroll
    for (int l = 0; l < N; l++) packed[l] = __ldg(reinterpret_cast<const uint32_t *>(U + l * plane + j * mp + i0));
    const int fj = f[j];
    double out[4];
#pragma unroll 1
    for (int s = 0; s < 4; s++) {
        if (i0 + s >= m) { out[s] = 0.0; continue; }
        uint32_t u[N];
#pragma unroll
        for (int l = 0; l < N; l++) u[l] = __byte_perm(packed[l], 0u, 0x4440 + s);
        uint64_t *cpp = WANT_CPP ? Cpp + ((size_t)j * m + i0 + s) * 4 : nullptr;
        double cij = crt_one<N>(u, e[i0 + s] + fj, cpp);
        double t = alpha * cij;
        double *dst = C + (i0 + s) + j * ldc;
        out[s] = (beta == 0.0) ? t : fma(beta, *dst, t);
    }
    double *dst = C + i0 + j * ldc;
    if (i0 + 3 < m && ((((uintptr_t)dst) & 15) == 0)) {
        reinterpret_cast<double2 *>(dst)[0] = make_double2(out[0], out[1]);
        reinterpret_cast<double2 *>(dst)[1] = make_double2(out[2], out[3]);
    } else {
        for (int s = 0; s < 4 && i0 + s < m; s++) dst[s] = out[s];
    }
}

template <int N>
int launch_n(int64_t m, int64_t n, const uint8_t *U, int64_t mp, const int32_t *e, const int32_t *f, double alpha,
             double beta, double *C, int64_t ldc, uint64_t *Cpp, cudaStream_t st)
{
    dim3 grid((unsigned)n, (unsigned)((m + 511) / 512));
    if (Cpp) k4_crt<N, true><<<grid, 128, 0, st>>>(m, n, U, mp, e, f, alpha, beta, C, ldc, Cpp);
    else k4_crt<N, false><<<grid, 128, 0, st>>>(m, n, U, mp, e, f, alpha, beta, C, ldc, nullptr);
    oz2_count_launches(1);
    return (int)cudaGetLastError();
}

} // namespace

int oz2_crt_upload_tables(const Oz2HostTables &t)
{
    OZ2_CUDA_TRY(cudaMemcpyToSymbol(c_crt, t.crt, sizeof(t.crt)));
    return 0;
}

int oz2_launch_crt(int N, int64_t m, int64_t n, const uint8_t *U, int64_t mp, const int32_t *e, const int32_t *f,
                   double alpha, double beta, double *C, int64_t ldc, uint64_t *Cpp, cudaStream_t st)
{
    if (m <= 0 || n <= 0) return 0;
    switch (N) {
#define OZ2_CASE(NN) case NN: return launch_n<NN>(m, n, U, mp, e, f, alpha, beta, C, ldc, Cpp, st);
        OZ2_CASE(2) OZ2_CASE(3) OZ2_CASE(4) OZ2_CASE(5) OZ2_CASE(6) OZ2_CASE(7) OZ2_CASE(8) OZ2_CASE(9)
        OZ2_CASE(10) OZ2_CASE(11) OZ2_CASE(12) OZ2_CASE(13) OZ2_CASE(14) OZ2_CASE(15) OZ2_CASE(16)
        OZ2_CASE(17) OZ2_CASE(18) OZ2_CASE(19) OZ2_CASE(20)
#undef OZ2_CASE
    }
    return -1;
}
