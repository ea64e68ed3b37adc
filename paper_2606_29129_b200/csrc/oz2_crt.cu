// oz2_crt.cu -- S4 + S5: CRT reconstruction and unscaling.
//
//   C'  = sum_l w_l U_l,  w_l = P_l q_l                       (eq. (2); Theorem 1)
//   C'' = rmod(C', P) in [-P/2, P/2)                           (eq. (3); reading R7)
//   C   = RN_64(C'') 2^-(e_i+f_j)                              (Step 4; reading R8)
//   out = alpha C (+ beta C_in)                                (reading R9)
//
// Everything up to the single rounding RN_64 is EXACT integer arithmetic (the weights have up to 156 bits, C' up
// to 169).  The sum over the moduli is a dense contraction and runs on the tensor cores (k5_crt_tc below: one
// tcgen05.mma kind::i8 per 128 elements over byte-sliced weights); the epilogue threads fold the byte slices into
// 32-bit words, estimate Q ~ C'/P in FP64 (|error| < 2^-30; the rare near-half cases take an exact compare
// against P/2), form C'' = C' - Q P in two's complement, and round a 64-bit normalised mantissa with a sticky
// bit once.  HBM traffic: N bytes in + 8 bytes out per element.
#include "oz2_common.cuh"
#include "oz2_tc.cuh"
#include <string.h>

namespace {

__constant__ Oz2CrtTab c_crt[OZ2_MAX_MODULI + 1];

// number of 32-bit words of P for N moduli (log2 P: 15.99, 23.98, 31.95, 39.9, ... 155.4)
__host__ __device__ constexpr int words_of_P(int N)
{
    return N <= 4 ? 1 : N <= 8 ? 2 : N <= 12 ? 3 : N <= 16 ? 4 : 5;
}

// RN of (mant64 | sticky) * 2^sc to a format with PB significand bits, subnormal quantum 2^QMIN and largest exponent
// EMAX (FP64: 53, -1074, 1023; FP32: 24, -149, 127), with a single rounding, subnormals and overflow included.
// The result is returned as a double (exact for both formats).
template <int PB, int QMIN, int EMAX>
__device__ __noinline__ double round_scaled_slow(unsigned long long mant, uint32_t sticky, int sc)
{
    // value in [2^(63+sc), 2^(64+sc))
    int Ex = 63 + sc;
    if (Ex > EMAX) return __longlong_as_double(0x7FF0000000000000ll);
    int rs = QMIN - sc;                           // bits dropped below the subnormal quantum
    if (rs < 64 - PB) rs = 64 - PB;               // never keep more than PB bits
    unsigned long long q, half, low;
    if (rs >= 65) return 0.0;
    if (rs == 64) { q = 0; half = mant >> 63; low = (mant << 1) | sticky; }
    else { q = mant >> rs; half = (mant >> (rs - 1)) & 1ull; low = (mant & ((1ull << (rs - 1)) - 1)) | sticky; }
    if (half && (low || (q & 1ull))) q += 1;
    // q * 2^(sc + rs)
    int qe = sc + rs;
    if (PB == 53 && qe == -1074) return __longlong_as_double((long long)q);   // FP64 subnormal (or the smallest normal)
    double d = (double)(long long)q;                                   // q <= 2^53: exact
    // qe > -1074 here means the result is normal; scale in two exact steps to stay in range
    int h1 = qe / 2, h2 = qe - h1;
    d *= __longlong_as_double((long long)(h1 + 1023) << 52);
    d *= __longlong_as_double((long long)(h2 + 1023) << 52);
    return d;
}

// C'' = rmod(C', P), RN_64(C'') 2^-esum from the words c[0..NW] of C' = sum_l w_l U_l (c[NW] < 2^13)
// TO = double: RN_64; TO = float: RN_32 of the same exact integer (SGEMM variant).
// crt_exact handles every case (near-half quotients, subnormal / overflowing results, the C'' words for the parity
// surface); crt_fast below is its branch-free common case and says when it does not apply.
template <int NW, typename TO>
__device__ __noinline__ TO crt_exact(const uint32_t (&c)[NW + 1], const Oz2CrtTab &T, int esum, uint64_t *cpp_out)
{
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
    if (ptop == 0ull) return (TO)0;
    const int lz = __clzll((long long)ptop);
    const unsigned long long mant = (ptop << lz) | ((pmid >> 1) >> (63 - lz));
    const uint32_t sticky = (((pmid << lz) | plow) != 0ull) ? 1u : 0u;
    const int pos = base + 63 - lz;                                   // |C''| in [2^pos, 2^(pos+1))
    const int sc = pos - 63 - esum;                                   // result = mant 2^sc
    const int Ex = pos - esum;
    if constexpr (sizeof(TO) == 8) {
        double v;
        if (Ex >= -1020 && Ex <= 1021) {
            const double d = __ull2double_rn(mant | sticky);          // the one rounding, ties to even
            v = __longlong_as_double(__double_as_longlong(d) + ((long long)sc << 52));
        } else {
            v = round_scaled_slow<53, -1074, 1023>(mant, sticky, sc);
        }
        return __longlong_as_double(__double_as_longlong(v) | (long long)(m64 << 63));
    } else {
        float v;
        if (Ex >= -124 && Ex <= 125) {
            const float d = __ull2float_rn(mant | sticky);            // the one rounding, ties to even
            v = __int_as_float(__float_as_int(d) + sc * 8388608);
        } else {
            v = (float)round_scaled_slow<24, -149, 127>(mant, sticky, sc);      // exact conversion
        }
        return __int_as_float(__float_as_int(v) | (int)((uint32_t)negm & 0x80000000u));
    }
}

// ---- multiword helpers: one PTX carry chain each (the C++ formulation costs about twice the instructions) ----------
// r = a - b over W words (borrow out of the top word is dropped)
template <int W>
__device__ __forceinline__ void mp_sub(uint32_t (&r)[W], const uint32_t (&a)[W], const uint32_t (&b)[W])
{
    static_assert(W >= 2 && W <= 6, "word count");
    if constexpr (W == 2)
        asm("sub.cc.u32 %0, %2, %4;\n\tsubc.u32 %1, %3, %5;" : "=r"(r[0]), "=r"(r[1]) : "r"(a[0]), "r"(a[1]), "r"(b[0]), "r"(b[1]));
    else if constexpr (W == 3)
        asm("sub.cc.u32 %0, %3, %6;\n\tsubc.cc.u32 %1, %4, %7;\n\tsubc.u32 %2, %5, %8;"
            : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]) : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(b[0]), "r"(b[1]), "r"(b[2]));
    else if constexpr (W == 4)
        asm("sub.cc.u32 %0, %4, %8;\n\tsubc.cc.u32 %1, %5, %9;\n\tsubc.cc.u32 %2, %6, %10;\n\tsubc.u32 %3, %7, %11;"
            : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
            : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]), "r"(b[2]), "r"(b[3]));
    else if constexpr (W == 5)
        asm("sub.cc.u32 %0, %5, %10;\n\tsubc.cc.u32 %1, %6, %11;\n\tsubc.cc.u32 %2, %7, %12;\n\tsubc.cc.u32 %3, %8, %13;\n\t"
            "subc.u32 %4, %9, %14;"
            : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4])
            : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(a[4]), "r"(b[0]), "r"(b[1]), "r"(b[2]), "r"(b[3]), "r"(b[4]));
    else
        asm("sub.cc.u32 %0, %6, %12;\n\tsubc.cc.u32 %1, %7, %13;\n\tsubc.cc.u32 %2, %8, %14;\n\tsubc.cc.u32 %3, %9, %15;\n\t"
            "subc.cc.u32 %4, %10, %16;\n\tsubc.u32 %5, %11, %17;"
            : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5])
            : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(a[4]), "r"(a[5]), "r"(b[0]), "r"(b[1]), "r"(b[2]), "r"(b[3]), "r"(b[4]),
              "r"(b[5]));
}
// x += one (one = 0 or 1) over W words
template <int W>
__device__ __forceinline__ void mp_inc(uint32_t (&x)[W], uint32_t one)
{
    static_assert(W >= 1 && W <= 5, "word count");
    if constexpr (W == 1) x[0] += one;
    else if constexpr (W == 2) asm("add.cc.u32 %0, %0, %2;\n\taddc.u32 %1, %1, 0;" : "+r"(x[0]), "+r"(x[1]) : "r"(one));
    else if constexpr (W == 3)
        asm("add.cc.u32 %0, %0, %3;\n\taddc.cc.u32 %1, %1, 0;\n\taddc.u32 %2, %2, 0;" : "+r"(x[0]), "+r"(x[1]), "+r"(x[2]) : "r"(one));
    else if constexpr (W == 4)
        asm("add.cc.u32 %0, %0, %4;\n\taddc.cc.u32 %1, %1, 0;\n\taddc.cc.u32 %2, %2, 0;\n\taddc.u32 %3, %3, 0;"
            : "+r"(x[0]), "+r"(x[1]), "+r"(x[2]), "+r"(x[3]) : "r"(one));
    else
        asm("add.cc.u32 %0, %0, %5;\n\taddc.cc.u32 %1, %1, 0;\n\taddc.cc.u32 %2, %2, 0;\n\taddc.cc.u32 %3, %3, 0;\n\taddc.u32 %4, %4, 0;"
            : "+r"(x[0]), "+r"(x[1]), "+r"(x[2]), "+r"(x[3]), "+r"(x[4]) : "r"(one));
}

// per-N constants of the common case; passed to the kernel by value (__grid_constant__), so that they are constant-bank
// operands of the instructions that use them and are never loaded
struct K5Consts {
    uint32_t Pn[OZ2_MAX_WORDS];     // 2^(32 NW) - P: C' + Q Pn = C' - Q P  (mod 2^(32 NW))
    uint32_t nterms;                // (unused padding)
    double K0, K1;                  // 2^(32 (NW-1)) / P and 2^(32 (NW-2)) / P: weights of the two top 32-bit columns
};
K5Consts h_k5[OZ2_MAX_MODULI + 1];                 // host copy, filled by oz2_crt_upload_tables

// The common case without a branch, straight from the byte slices S[0 .. 4 NW) of one element:
//   Z_k  : the 32-bit columns of C' before carries, sum_b S[4k+b] 256^b (< 2^46) up to the pairing below; C' = sum_k Z_k 2^(32 k)
//   Q    = round(C' / P) from the two top columns in FP64 (dropped columns < 2^-22.9, arithmetic < 2^-38: any Q within
//          2^-20 of a half-integer is handed to the exact routine)
//   R    = C' + Q (2^(32 NW) - P) mod 2^(32 NW) = C'' in two's complement: W_k = Z_k + Q Pn_k (< 2^47) per column, then
//          ONE carry chain over the NW columns -- fold and subtraction together cost 5 instructions per word
//   |R|  -> the 64 bits from the leading one (top three words after at most NW - 3 whole-word shifts; a value below
//          2^64 passes exactly through the clamped funnel shifts) + sticky bit -> one rounding (I2F) -> exponent field
// `rare` is set when the result needs crt_exact (near-half quotient, subnormal or overflowing result).
template <int NW, typename TO>
__device__ __forceinline__ TO crt_fast(const uint32_t *S, const K5Consts &T, int esum, bool &rare)
{
    // (the low halves a_k travel in pairs: Z_k carries a_k + 2^32 a_(k+1) as the 64-bit addend of its multiply-add and
    // Z_(k+1) = 2^16 b_(k+1) none, so that no addend needs a zeroed high word; sum_k Z_k 2^(32 k) is unchanged)
    uint32_t a[NW], b[NW];
#pragma unroll
    for (int k = 0; k < NW; k++) {
        a[k] = S[4 * k] + (S[4 * k + 1] << 8);                        // < 2^30
        b[k] = S[4 * k + 2] + (S[4 * k + 3] << 8);
    }
    unsigned long long Z[NW];
#pragma unroll
    for (int k = NW - 2; k >= 0; k -= 2) {
        Z[k] = (unsigned long long)b[k] * 65536ull + (((unsigned long long)a[k + 1] << 32) | a[k]);
        Z[k + 1] = (unsigned long long)b[k + 1] * 65536ull;
    }
    if constexpr (NW & 1) Z[0] = (unsigned long long)b[0] * 65536ull + (unsigned long long)a[0];
    // ---- Q (Z < 2^63; the conversion of the second column may round: relative 2^-53, far below the guard)
    double qd = (double)(long long)Z[NW - 1] * T.K0;
    if constexpr (NW >= 2) qd = fma((double)(long long)Z[NW - 2], T.K1, qd);
    const double MAGIC = 6755399441055744.0;                          // 1.5 2^52: RN to an integer in the low word
    const double tq = qd + MAGIC;
    const uint32_t Q = (uint32_t)__double2loint(tq);
    rare = fabs(qd - (tq - MAGIC)) > 0.5 - 9.5367431640625e-07;       // within 2^-20 of a half-integer: exact compare needed
    // ---- R = C' - Q P (mod 2^(32 NW))
    uint32_t r[NW];
    {
        unsigned long long W[NW];
#pragma unroll
        for (int k = 0; k < NW; k++) W[k] = (unsigned long long)Q * T.Pn[k] + Z[k];
        uint32_t lo[NW], hi[NW];
#pragma unroll
        for (int k = 0; k < NW; k++) { lo[k] = (uint32_t)W[k]; hi[k] = (uint32_t)(W[k] >> 32); }
        r[0] = lo[0];
        if constexpr (NW == 2) r[1] = lo[1] + hi[0];
        if constexpr (NW == 3)
            asm("add.cc.u32 %0, %2, %3;\n\taddc.u32 %1, %4, %5;" : "=r"(r[1]), "=r"(r[2]) : "r"(lo[1]), "r"(hi[0]), "r"(lo[2]), "r"(hi[1]));
        if constexpr (NW == 4)
            asm("add.cc.u32 %0, %3, %4;\n\taddc.cc.u32 %1, %5, %6;\n\taddc.u32 %2, %7, %8;"
                : "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(lo[1]), "r"(hi[0]), "r"(lo[2]), "r"(hi[1]), "r"(lo[3]), "r"(hi[2]));
        if constexpr (NW == 5)
            asm("add.cc.u32 %0, %4, %5;\n\taddc.cc.u32 %1, %6, %7;\n\taddc.cc.u32 %2, %8, %9;\n\taddc.u32 %3, %10, %11;"
                : "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4])
                : "r"(lo[1]), "r"(hi[0]), "r"(lo[2]), "r"(hi[1]), "r"(lo[3]), "r"(hi[2]), "r"(lo[4]), "r"(hi[3]));
    }
    // ---- |R| (|C''| <= P/2 < 2^(32 NW - 1)), branch-free negate
    const uint32_t negm = (uint32_t)((int32_t)r[NW - 1] >> 31);
    uint32_t x[NW];
#pragma unroll
    for (int t = 0; t < NW; t++) x[t] = r[t] ^ negm;
    mp_inc<NW>(x, negm & 1u);
    // ---- 64-bit mantissa from the leading one + sticky bit; value = mant 2^sc
    unsigned long long mant;
    int sc = -esum;
    if constexpr (NW == 1) mant = x[0];
    else if constexpr (NW == 2) mant = ((unsigned long long)x[1] << 32) | x[0];
    else {
        sc += 32 * (NW - 2);
#pragma unroll
        for (int s = 0; s < NW - 3; s++) {                            // whole-word shifts while the top word is empty
            const bool z = x[NW - 1] == 0u;
#pragma unroll
            for (int t = NW - 1; t >= 1; t--) x[t] = z ? x[t - 1] : x[t];
            x[0] = z ? 0u : x[0];
            sc -= z ? 32 : 0;
        }
        const int lz = __clz((int)x[NW - 1]);                         // 32 for an empty top word: the shifts below clamp
        const uint32_t mh = __funnelshift_lc(x[NW - 2], x[NW - 1], lz), ml = __funnelshift_lc(x[NW - 3], x[NW - 2], lz);
        uint32_t rest = __funnelshift_lc(0u, x[NW - 3], lz);
#pragma unroll
        for (int t = 0; t < NW - 3; t++) rest |= x[t];
        mant = ((unsigned long long)mh << 32) | (ml | (rest != 0u ? 1u : 0u));
        sc -= lz;
    }
    if constexpr (sizeof(TO) == 8) {
        const double d = NW == 1 ? (double)(uint32_t)mant : __ull2double_rn(mant);   // the one rounding, ties to even
        const int hd = __double2hiint(d);
        const bool zero = hd == 0;
        const int be = (hd >> 20) + sc;                               // biased exponent of the result
        rare |= !zero && (uint32_t)(be - 2) > 2043u;                  // subnormal or overflowing result: exact routine
        const int hw = (hd + (sc << 20)) | (int)(negm & 0x80000000u);
        return __hiloint2double(zero ? 0 : hw, __double2loint(d));
    } else {
        const float d = NW == 1 ? __uint2float_rn((uint32_t)mant) : __ull2float_rn(mant);
        const int hd = __float_as_int(d);
        const bool zero = hd == 0;
        const int be = (hd >> 23) + sc;
        rare |= !zero && (uint32_t)(be - 2) > 251u;
        const int bits = (hd + (sc << 23)) | (int)(negm & 0x80000000u);
        return __int_as_float(zero ? 0 : bits);
    }
}

// by-value gate to crt_exact for the parity surface (every element, C'' words wanted): the words travel in a struct
// so that the caller keeps them in registers
template <int NW>
struct CWords { uint32_t w[NW + 1]; };
template <int NW, typename TO>
__device__ __noinline__ TO crt_exact_v(CWords<NW> cw, int N, int esum, uint64_t *cpp_out)
{
    return crt_exact<NW, TO>(cw.w, c_crt[N], esum, cpp_out);
}

// The rare path of the production kernel, decoupled from the registers of the common case: C' = sum_l w_l U_l is
// recomputed in plain integer arithmetic from the element's N residue bytes in global memory (planes `plane` bytes
// apart), then crt_exact.
template <int NW, typename TO>
__device__ __noinline__ TO crt_exact_global(const uint8_t *__restrict__ Uel, size_t plane, int N, int esum)
{
    uint32_t c[NW + 1];
#pragma unroll
    for (int t = 0; t <= NW; t++) c[t] = 0u;
    for (int l = 0; l < N; l++) {
        const uint32_t u = Uel[(size_t)l * plane];
        unsigned long long carry = 0;
#pragma unroll
        for (int t = 0; t < NW; t++) {
            const unsigned long long v = (unsigned long long)u * c_crt[N].w[l][t] + c[t] + carry;
            c[t] = (uint32_t)v;
            carry = v >> 32;
        }
        c[NW] += (uint32_t)carry;
    }
    return crt_exact<NW, TO>(c, c_crt[N], esum, nullptr);
}

// =============================================================================================
// Tensor-core CRT.  sum_l w_l U_l is itself a small dense contraction: with the weights cut into bytes,
//     S[i][t] = sum_l U_l[i] * byte_t(w_l),   t = 0 .. 4 NW - 1,      C'[i] = sum_t S[i][t] 256^t,
// i.e. (128 elements) x (K = moduli, zero padded to 32) x (16 or 32 byte slices): ONE tcgen05.mma kind::i8 per 128
// elements (unsigned x unsigned, S < 2^21).  A = the U planes as they lie in memory ([l][j][i], i fastest) fetched
// by TMA as an MN-major SWIZZLE_128B operand (planes >= N are zero filled by the TMA bounds check); B = a constant
// 0.5 / 1 KB image of the weight bytes in shared memory (K-major, no swizzle).  This replaces 4 NW N wide
// multiply-adds per element on the integer pipe; the epilogue threads (one element each) only fold the slices
// into words and run crt_from_words.
// =============================================================================================
constexpr int K5_STAGES = 3, K5_NBUF = 2, K5_THREADS = 320;     // warps: TMA, MMA, 2 sets of 4 epilogue warps
constexpr int K5_TILE_I = 512, K5_KPAD = 32;                    // one pipeline step = 4 MMAs of 128 elements
constexpr int K5_STAGE_BYTES = K5_TILE_I * K5_KPAD;             // 16 KB
constexpr int K5_SMEM = K5_STAGES * K5_STAGE_BYTES + 1024 /*B image*/ + 1024 /*alignment*/ + 512 /*barriers*/;

__device__ uint8_t g_wb_image[OZ2_MAX_MODULI + 1][1024];        // per N: B operand image (see upload)

// fold the byte slices S[0 .. 4 NW) of one element into the words of C'
template <int NW>
__device__ __forceinline__ void k5_fold(const uint32_t *S, uint32_t (&c)[NW + 1])
{
    unsigned long long carry = 0;
#pragma unroll
    for (int k = 0; k < NW; k++) {       // V_k = sum_{b<4} S[4k+b] 256^b (< 2^46), then carries
        unsigned long long v = (unsigned long long)S[4 * k] + ((unsigned long long)S[4 * k + 1] << 8) +
                               ((unsigned long long)S[4 * k + 2] << 16) + ((unsigned long long)S[4 * k + 3] << 24) + carry;
        c[k] = (uint32_t)v;
        carry = v >> 32;
    }
    c[NW] = (uint32_t)carry;
}

template <bool BETA0, typename TO>
__device__ __forceinline__ void k5_store(TO cij, TO alpha, TO beta, TO *dst)
{
    if constexpr (sizeof(TO) == 8) {
        const double tt = alpha * cij;
        *dst = (BETA0 || beta == 0.0) ? tt : fma(beta, *dst, tt);
    } else {
        const float tt = __fmul_rn(alpha, cij);
        *dst = (BETA0 || beta == 0.0f) ? tt : __fmaf_rn(beta, *dst, tt);
    }
}

// the two elements (i, j) and (i + 128, j) of one thread: C'' -> C -> alpha / beta -> store.  Both go through the
// branch-free crt_fast side by side (two independent dependency chains per thread); the exact routine is the rare path.
template <int NW, bool WANT_CPP, bool BETA0, typename TO>
__device__ __forceinline__ void k5_finish2(const uint32_t *Sa, const uint32_t *Sb, const K5Consts &T, int N, bool ok_b, int esum_a, int esum_b, TO alpha,
                                           TO beta, TO *__restrict__ C, int ldc, uint64_t *__restrict__ Cpp, int m,
                                           const uint8_t *__restrict__ U, int mp, size_t plane, int i, int j)
{
    TO va, vb;
    if constexpr (WANT_CPP) {
        uint64_t *cpp = Cpp + ((size_t)j * m + i) * 4;
        CWords<NW> wa, wb;
        k5_fold<NW>(Sa, wa.w);
        k5_fold<NW>(Sb, wb.w);
        va = crt_exact_v<NW, TO>(wa, N, esum_a, cpp);
        vb = ok_b ? crt_exact_v<NW, TO>(wb, N, esum_b, cpp + 128 * 4) : (TO)0;
    } else {
        bool rare_a, rare_b;
        va = crt_fast<NW, TO>(Sa, T, esum_a, rare_a);
        vb = crt_fast<NW, TO>(Sb, T, esum_b, rare_b);
        if (rare_a || (rare_b && ok_b)) {                             // rare: near-half quotient, subnormal or overflowing result
            const uint8_t *Uel = U + ((size_t)j * (size_t)mp + (size_t)i);
            if (rare_a) va = crt_exact_global<NW, TO>(Uel, plane, N, esum_a);
            if (rare_b && ok_b) vb = crt_exact_global<NW, TO>(Uel + 128, plane, N, esum_b);
        }
    }
    TO *dst = C + ((int64_t)j * ldc + i);
    k5_store<BETA0, TO>(va, alpha, beta, dst);
    if (ok_b) k5_store<BETA0, TO>(vb, alpha, beta, dst + 128);
}

// One pipeline step = a tile of 512 consecutive elements of one column of C: four TMA boxes (128 elements x 32 planes)
// in one 16 KB stage, four MMAs into one accumulator buffer of 4 NS columns.  The two epilogue sets take every second
// tile of the CTA; a thread owns the four elements il + 128 h of its tile and works through them as two pairs, so that
// the barrier wait, the tile walk, f_j and the address arithmetic are paid once per four elements.  Each set has ONE
// accumulator buffer: it is handed back as soon as the second pair has been read out of tensor memory, i.e. half a
// tile of epilogue work before the set needs the next one.
template <int NW, bool WANT_CPP, bool BETA0, typename TO>
__global__ void __launch_bounds__(K5_THREADS, NW <= 4 ? 3 : 2)
k5_crt_tc(const __grid_constant__ CUtensorMap mapU, int N, int m, int n, const int32_t *__restrict__ e,
          const int32_t *__restrict__ f, TO alpha, TO beta, TO *__restrict__ C, int ldc,
          uint64_t *__restrict__ Cpp, const uint8_t *__restrict__ U, int mp, const __grid_constant__ K5Consts T, int ib0, int nib)
{
    constexpr int NS = NW <= 4 ? 16 : 32;                    // byte slices = MMA N
    constexpr int BUF_COLS = 4 * NS;                         // four 128-element MMAs per accumulator buffer
    // kind::i8 instruction descriptor: D = S32, A = B = unsigned 8 bit, A MN-major, B K-major, N = NS, M = 128
    constexpr uint32_t IDESC = (2u << 4) | (1u << 15) | ((uint32_t)(NS >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem0 = (smem_u32(smem_raw) + 1023u) & ~1023u;           // shared-space addresses from here on
    const uint32_t wb = smem0 + K5_STAGES * K5_STAGE_BYTES;
    const uint32_t full = wb + 1024, empty = full + 8 * K5_STAGES, tfull = empty + 8 * K5_STAGES, tempty = tfull + 8 * K5_NBUF;
    const uint32_t tmem_slot = tempty + 8 * K5_NBUF;
    uint8_t *gen0 = smem_raw + (smem0 - smem_u32(smem_raw));                // generic pointer to the aligned base

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // The grid is nib x gj CTAs: CTA b owns row block ib = ib0 + b % nib (512 rows: its exponents e_i stay in registers) and
    // walks the columns j = b / nib, + gj, + 2 gj, ...
    const int gj = (int)gridDim.x / nib;
    const int j0 = (int)blockIdx.x / nib, ib = ib0 + ((int)blockIdx.x - j0 * nib);

    if (threadIdx.x == 0) {
        for (int s = 0; s < K5_STAGES; s++) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(full + 8 * s));
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(empty + 8 * s));
        }
        for (int b = 0; b < K5_NBUF; b++) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(tfull + 8 * b));
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 4;" ::"r"(tempty + 8 * b));
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&mapU) : "memory");
    }
    // B operand image: generic-proxy writes, then made visible to the async (tensor core) proxy
    for (int t = threadIdx.x; t < 1024 / 16; t += K5_THREADS)
        reinterpret_cast<uint4 *>(gen0 + K5_STAGES * K5_STAGE_BYTES)[t] = reinterpret_cast<const uint4 *>(g_wb_image[N])[t];
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "n"(K5_NBUF * BUF_COLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    uint32_t tmem_base;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));
    pdl_launch_dependents();                      // only now: this CTA owns its tensor-memory columns (oz2_common.cuh)
    pdl_wait();                                   // the residue products come from the GEMM

    if (warp == 0) {
        if (lane == 0) {
            int s = 0; uint32_t ph = 0;
            for (int j = j0; j < n; j += gj) {
                mbar_wait_idle(empty + 8 * s, ph ^ 1u);          // the epilogue paces this kernel: poll lazily
                mbar_expect_tx_a(full + 8 * s, K5_STAGE_BYTES);
                const uint32_t dst = smem0 + s * K5_STAGE_BYTES;
#pragma unroll
                for (int h = 0; h < 4; h++)                      // boxes past the end of the column are zero filled
                    tma_load_3d_a(&mapU, full + 8 * s, dst + h * (K5_STAGE_BYTES / 4), ib * K5_TILE_I + 128 * h, j, 0);
                if (++s == K5_STAGES) { s = 0; ph ^= 1u; }
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            int s = 0, b = 0; uint32_t ph = 0, bph = 0;
            // B: K-major, no swizzle: core matrices 8 rows x 16 B; K-direction stride (LBO) 128 B, 8-row groups (SBO) 256 B
            const uint64_t bdesc = (uint64_t)((wb & 0x3FFFFu) >> 4) | ((uint64_t)(128u >> 4) << 16) |
                                   ((uint64_t)(256u >> 4) << 32) | (1ull << 46);
            // A: MN-major, SWIZZLE_128B: one 128-byte MN block per K row, 8-row K groups 1024 B apart (SBO)
            const uint64_t adesc0 = ((uint64_t)1 << 16) | ((uint64_t)(1024u >> 4) << 32) | (1ull << 46) | (2ull << 61);
            for (int j = j0; j < n; j += gj) {
                mbar_wait_a(tempty + 8 * b, bph ^ 1u);
                mbar_wait_idle(full + 8 * s, ph);
                tc_fence_after();
                const uint32_t sa = smem0 + s * K5_STAGE_BYTES;
#pragma unroll
                for (int h = 0; h < 4; h++)
                    tc_mma_i8(tmem_base + (uint32_t)(b * BUF_COLS + h * NS),
                              adesc0 | (uint64_t)(((sa + h * (K5_STAGE_BYTES / 4)) & 0x3FFFFu) >> 4), bdesc, IDESC, 0u);
                tc_commit_a(empty + 8 * s);
                tc_commit_a(tfull + 8 * b);
                if (++s == K5_STAGES) { s = 0; ph ^= 1u; }
                if (++b == K5_NBUF) { b = 0; bph ^= 1u; }
            }
        }
    } else {
        const int q = warp & 3;                              // TMEM lane quarter of this warp
        const int set = (warp - 2) >> 2;                     // epilogue set 0 / 1 takes every second tile of the CTA
        uint32_t bph = 0;
        const uint32_t bar_full = tfull + 8 * set, bar_empty = tempty + 8 * set;
        // this set takes the columns j0 + set gj, + 2 gj, ...
        const int stride = 2 * gj;
        const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(set * BUF_COLS);
        const int i = ib * K5_TILE_I + q * 32 + lane;        // first of the four rows i + 128 h of this thread
        const size_t plane = (size_t)n * (size_t)mp;
        int ev[4];
#pragma unroll
        for (int h = 0; h < 4; h++) ev[h] = i + 128 * h < m ? __ldg(e + i + 128 * h) : 0;
        int j = j0 + set * gj;
        int fnext = j < n ? __ldg(f + j) : 0;                // f_j of the tile about to be processed, loaded one tile ahead
        for (; j < n; j += stride) {
            const int jcur = j;
            const int fj = fnext;
            if (j + stride < n) fnext = __ldg(f + j + stride);
            mbar_wait_a(bar_full, bph);
            bph ^= 1u;
            tc_fence_after();
#pragma unroll
            for (int pr = 0; pr < 2; pr++) {                 // elements (i + 256 pr, i + 256 pr + 128)
                uint32_t S[2 * NS];
                tc_ld32_nowait(taddr + (uint32_t)(pr * 2 * NS), *reinterpret_cast<uint32_t(*)[32]>(S));
                if constexpr (NS == 32) tc_ld32_nowait(taddr + (uint32_t)(pr * 2 * NS + 32), *reinterpret_cast<uint32_t(*)[32]>(S + 32));
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                if (pr == 1) {                               // both pairs are out of tensor memory: hand the buffer back
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive_a(bar_empty);
                }
                const int ia = i + 256 * pr;
                if (ia < m)
                    k5_finish2<NW, WANT_CPP, BETA0, TO>(S, S + NS, T, N, ia + 128 < m, ev[2 * pr] + fj, ev[2 * pr + 1] + fj, alpha, beta, C, ldc,
                                                        Cpp, m, U, mp, plane, ia, jcur);
            }
        }
    }
    __syncthreads();
    if (warp == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(K5_NBUF * BUF_COLS) : "memory");
}

template <int NW, typename TO>
int launch_tc(int N, int64_t m, int64_t n, const uint8_t *U, int64_t mp, const int32_t *e, const int32_t *f, TO alpha,
              TO beta, TO *C, int64_t ldc, uint64_t *Cpp, cudaStream_t st)
{
    // U planes [N][n][mp] -> 3-D map (i, j, l), box (128, 1, 32): rows i >= mp and planes l >= N are zero filled
    CUtensorMap map;
    const TensorMapKey key = { U, (uint64_t)mp, (uint64_t)n, (uint64_t)N, (uint64_t)mp, (uint64_t)(n * mp),
                               128u, 1u, (uint32_t)K5_KPAD, (uint32_t)CU_TENSOR_MAP_SWIZZLE_128B };
    const int erc = encode_u8_3d_cached(&map, key);
    if (erc) return erc;
    const int sms = oz2_num_sms();
    const int64_t tiles_i = (m + K5_TILE_I - 1) / K5_TILE_I;
    const int per_sm = NW <= 4 ? 3 : 2;                   // TMEM: 128 / 256 columns per CTA; 320 threads; 3 x 51 KB shared
    const int64_t gmax = (int64_t)sms * per_sm;
    if (ldc >= (int64_t)1 << 31 || mp >= (int64_t)1 << 31) return (int)cudaErrorInvalidValue;
    const int mi = (int)m, ni = (int)n, ldi = (int)ldc, mpi = (int)mp;
    // (the > 48 KB dynamic shared memory opt-in of these kernels is per device: oz2_crt_upload_tables)
    auto launch = [&](auto kern, uint64_t *cpp) -> int {
        // grid = (row blocks of the launch) x (columns in flight); more row blocks than resident CTAs: several launches
        for (int64_t ib0 = 0; ib0 < tiles_i; ib0 += gmax) {
            const int64_t nib = tiles_i - ib0 < gmax ? tiles_i - ib0 : gmax;
            int64_t gj = gmax / nib;
            if (gj > n) gj = n;
            OZ2_CUDA_TRY(oz2_launch(kern, dim3((unsigned)(nib * gj)), dim3(K5_THREADS), K5_SMEM, st, map, N, mi, ni, e, f, alpha, beta, C, ldi, cpp,
                                    U, mpi, h_k5[N], (int)ib0, (int)nib));
            oz2_count_launches(1);
        }
        return 0;
    };
    int lrc;
    if (Cpp) lrc = launch(k5_crt_tc<NW, true, false, TO>, Cpp);
    else if (beta == (TO)0) lrc = launch(k5_crt_tc<NW, false, true, TO>, nullptr);
    else lrc = launch(k5_crt_tc<NW, false, false, TO>, nullptr);
    if (lrc) return lrc;
    return (int)cudaGetLastError();
}

// k5_crt_tc needs more than 48 KB of dynamic shared memory; the opt-in is a per-device attribute of each instantiation
template <int NW, typename TO>
int k5_opt_in_smem()
{
    OZ2_CUDA_TRY(cudaFuncSetAttribute(k5_crt_tc<NW, true, false, TO>, cudaFuncAttributeMaxDynamicSharedMemorySize, K5_SMEM));
    OZ2_CUDA_TRY(cudaFuncSetAttribute(k5_crt_tc<NW, false, true, TO>, cudaFuncAttributeMaxDynamicSharedMemorySize, K5_SMEM));
    OZ2_CUDA_TRY(cudaFuncSetAttribute(k5_crt_tc<NW, false, false, TO>, cudaFuncAttributeMaxDynamicSharedMemorySize, K5_SMEM));
    return 0;
}
template <typename TO>
int k5_opt_in_smem_all()
{
    int rc;
    if ((rc = k5_opt_in_smem<1, TO>())) return rc;
    if ((rc = k5_opt_in_smem<2, TO>())) return rc;
    if ((rc = k5_opt_in_smem<3, TO>())) return rc;
    if ((rc = k5_opt_in_smem<4, TO>())) return rc;
    return k5_opt_in_smem<5, TO>();
}

} // namespace

// runs once per device (ensure_device, under its lock) with that device current
int oz2_crt_upload_tables(const Oz2HostTables &t)
{
    int arc;
    if ((arc = k5_opt_in_smem_all<double>())) return arc;
    if ((arc = k5_opt_in_smem_all<float>())) return arc;
    OZ2_CUDA_TRY(cudaMemcpyToSymbol(c_crt, t.crt, sizeof(t.crt)));
    // B operand images of k5_crt_tc: element (slice s, modulus l) at (s/8) 256 + (l/16) 128 + (s%8) 16 + (l%16)
    static uint8_t img[OZ2_MAX_MODULI + 1][1024];
    memset(img, 0, sizeof(img));
    for (int N = 2; N <= OZ2_MAX_MODULI; N++)
        for (int l = 0; l < N; l++)
            for (int sl = 0; sl < 4 * OZ2_MAX_WORDS && sl < 32; sl++) {
                const uint8_t byte = (uint8_t)(t.crt[N].w[l][sl / 4] >> (8 * (sl % 4)));
                img[N][(sl / 8) * 256 + (l / 16) * 128 + (sl % 8) * 16 + (l % 16)] = byte;
            }
    OZ2_CUDA_TRY(cudaMemcpyToSymbol(g_wb_image, img, sizeof(img)));
    // constants of the common case: Pn = 2^(32 NW) - P, K0 = 2^(32 (NW - 1)) / P, K1 = K0 2^-32
    // (host copy: written by the first device's set-up only -- a later device's must not disturb launches on the first)
    static bool h_k5_ready = false;
    K5Consts *k5 = h_k5;
    for (int N = 2; N <= OZ2_MAX_MODULI && !h_k5_ready; N++) {
        const int nw = words_of_P(N);
        unsigned long long borrow = 0;
        for (int w = 0; w < nw; w++) {                       // 0 - P over nw words
            const unsigned long long d = 0ull - (unsigned long long)t.crt[N].P[w] - borrow;
            k5[N].Pn[w] = (uint32_t)d;
            borrow = (d >> 32) & 1ull;
        }
        k5[N].K0 = t.crt[N].invP;
        k5[N].K1 = t.crt[N].invP * 2.3283064365386963e-10;
    }
    h_k5_ready = true;
    return 0;
}

template <typename TO>
static int launch_crt_t(int N, int64_t m, int64_t n, const uint8_t *U, int64_t mp, const int32_t *e, const int32_t *f,
                        TO alpha, TO beta, TO *C, int64_t ldc, uint64_t *Cpp, cudaStream_t st)
{
    switch (words_of_P(N)) {
        case 1: return launch_tc<1, TO>(N, m, n, U, mp, e, f, alpha, beta, C, ldc, Cpp, st);
        case 2: return launch_tc<2, TO>(N, m, n, U, mp, e, f, alpha, beta, C, ldc, Cpp, st);
        case 3: return launch_tc<3, TO>(N, m, n, U, mp, e, f, alpha, beta, C, ldc, Cpp, st);
        case 4: return launch_tc<4, TO>(N, m, n, U, mp, e, f, alpha, beta, C, ldc, Cpp, st);
        default: return launch_tc<5, TO>(N, m, n, U, mp, e, f, alpha, beta, C, ldc, Cpp, st);
    }
}

int oz2_launch_crt(int N, int f32, int64_t m, int64_t n, const uint8_t *U, int64_t mp, const int32_t *e, const int32_t *f,
                   double alpha, double beta, void *C, int64_t ldc, uint64_t *Cpp, cudaStream_t st)
{
    if (m <= 0 || n <= 0) return 0;
    if (N < 2 || N > OZ2_MAX_MODULI) return -1;
    if (f32) return launch_crt_t<float>(N, m, n, U, mp, e, f, (float)alpha, (float)beta, static_cast<float *>(C), ldc, Cpp, st);
    return launch_crt_t<double>(N, m, n, U, mp, e, f, alpha, beta, static_cast<double *>(C), ldc, Cpp, st);
}
