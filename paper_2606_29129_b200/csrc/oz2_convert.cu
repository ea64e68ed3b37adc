// oz2_convert.cu -- S2: A' = trunc(diag(mu) A), B' = trunc(B diag(nu)) (Step 2) and the symmetric
// INT8 residues rmod(., p_l) for all N moduli in ONE pass over A and B.
//
// The reduction of an up-to-84-bit integer modulo N small moduli is a dense contraction, so it runs on the tensor
// cores: with d_i the base-256 digits of a non-negative image a'' of a',
//     a'' = sum_i d_i 256^i      =>      a'' mod p_l  =  ( sum_i d_i (256^i mod p_l) ) mod p_l ,
// i.e. (elements x digits) x (digits x moduli).  One tcgen05.mma kind::i8 (unsigned x unsigned, M = 128, K = 32,
// N = up to 64) handles 128 "quads" = 512 elements: a K row of 32 bytes carries the 8-byte digit strings of the 4
// consecutive elements of a quad side by side, and the B operand is a constant block-diagonal image of the byte
// weights 256^i mod p_l, so that accumulator column (l, slot) holds  Y = sum_i d_i(slot) (256^i mod p_l) < 2^20.
// When |a'| needs more than 63 bits (N >= 17, accurate mode from N = 15) a second K row carries digits 8 .. 11 and a
// second MMA with the weights 256^(8+i) mod p_l accumulates onto the same columns.  One more MMA with a constant
// all-ones operand adds a per-modulus bias.  What is left for the CUDA cores is 2 multiplies per element and modulus and a packed store:
//     a''  = a' + 2^63 (two's complement of a' with the top bit flipped: non-negative, sign handled for free;
//            2^95 in the wide format),
//     bias = (p-1)/2 - 2^63 mod p,  Y ~ a' + (p-1)/2 (mod p),  u = Y mod p = Y - umulhi(Y, magic) p  in [0, p),
//     r    = u - (p-1)/2  in [-(p-1)/2, (p-1)/2]  is the symmetric residue (reading R5 for p = 256, where the
//     byte is simply the low byte of a'); four u bytes are packed, the per-byte offset 128 - (p-1)/2 is added to the
//     packed word (no carries: u + 128 - (p-1)/2 <= 255) and 0x80808080 is XORed to give the four INT8 values.
// trunc(a 2^e) is one exponent-field addition and one FP64 -> INT64 conversion (round toward zero, exact because
// |a'| < 2^63); subnormal inputs and the wide (N >= 17 or accurate-mode) format take integer shifts.
//
// Data movement (the stage is bound by HBM traffic 8 + N bytes per element).  Planes are [l][row][kp], k fastest
// (K-major for the GEMM), kp = round_up(k, 128), zero padded.  A thread owns a quad (4 consecutive h of one vector)
// from the global load to the 4-byte store, so a warp stores 128 contiguous bytes per modulus.
//   * contiguous vectors (columns of B, or rows of A^T): 32-byte loads straight from global memory;
//   * strided vectors (rows of a column-major A): a CTA brings 16 rows x 128 h into shared memory with cp.async
//     (128-byte coalesced reads along the rows, transposed on the way in), refilled while the last round computes.
// The same two movers, without the tensor-core part, serve accurate mode's Abar / Bbar = ceil(mu' |.|).
#include "oz2_common.cuh"
#include "oz2_tc.cuh"

namespace {

// eq. (14), P:252-255 as compile-time constants (the epilogue is fully unrolled over the moduli)
__host__ __device__ constexpr uint32_t modulus_of(int l)
{
    constexpr uint32_t t[OZ2_MAX_MODULI] = OZ2_MODULI_LIST;
    return t[l];
}

constexpr int CV_THREADS = 128;                    // one MMA tile row (quad) per thread
constexpr int CV_TILE_BYTES = 128 * 32;            // A operand: 128 rows x 32 K bytes
constexpr int CV_IMG_BYTES = 64 * 32;              // B operand: 64 columns x 32 K bytes
constexpr int CV_ONES_BYTES = 256;                 // all-ones A operand of the bias MMA: one 8-row group, re-read for all 16 (SBO = 0)
constexpr int CV_TMEM_COLS = 64;
constexpr int CV_CHUNK_H = 4 * CV_THREADS;         // contiguous side: h per round

// operand images in the canonical no-swizzle K-major layout (see tile_off), 64 accumulator columns (= 16 moduli x 4
// slots) each.  [g][t]: column group g (moduli 16 g .. 16 g + 15), t = 0: weights of digits 0 .. 7, 1: weights of
// digits 8 .. 11 (wide format), 2: bias of the narrow format, 3: bias of the wide format.
__device__ uint8_t g_conv_img[2][4][CV_IMG_BYTES];

// byte offset of (row r, K byte kb) in a K-major, no-swizzle operand: 8 x 16-byte core matrices,
// K-direction core-matrix stride (LBO) 128 B, 8-row group stride (SBO) 256 B
__host__ __device__ constexpr int tile_off(int r, int kb) { return (r >> 3) * 256 + (kb >> 4) * 128 + (r & 7) * 16 + (kb & 15); }

__device__ __forceinline__ uint64_t kmajor_desc(uint32_t saddr, uint32_t sbo)
{
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(128u >> 4) << 16) | ((uint64_t)(sbo >> 4) << 32) | (1ull << 46);
}

// ---------------------------------------------------------------------------------------------
// trunc(a 2^ex)
// ---------------------------------------------------------------------------------------------
// zero / subnormal input (rare): integer shifts of the 52-bit mantissa; value = +-M 2^(ex - 1074)
__device__ __noinline__ long long trunc_subnormal(long long bits, int ex)
{
    const unsigned long long M = (unsigned long long)bits & 0x000FFFFFFFFFFFFFull;
    const int sh = ex - 1074;
    unsigned long long mag;
    if (sh >= 0) mag = M << (sh > 63 ? 63 : sh);
    else mag = (-sh < 64) ? (M >> (-sh)) : 0ull;
    return bits < 0 ? -(long long)mag : (long long)mag;
}

// narrow format: |a'| < 2^63.  Returns a' + 2^63 as an unsigned 64-bit integer (its bytes are the 8 digits).
__device__ __forceinline__ unsigned long long digits_narrow(double a, int ex)
{
    const long long bits = __double_as_longlong(a);
    const int hi = (int)(bits >> 32);
    const int be = (hi >> 20) & 0x7FF;
    long long t;
    if (be == 0) {
        t = (bits << 1) == 0 ? 0ll : trunc_subnormal(bits, ex);
    } else {
        const int ne = be + ex;                                   // biased exponent of a 2^ex
        const double x = __hiloint2double(hi + ex * 1048576, (int)bits);
        t = ne < 1023 ? 0ll : __double2ll_rz(x);                  // |a 2^ex| < 1 truncates to 0; else exact (< 2^63)
    }
    return (unsigned long long)t ^ 0x8000000000000000ull;
}

// wide format: |a'| < 2^95 as three 32-bit words of a' + 2^95 (two's complement, top bit flipped).
// Integer route (any input; used for zero / subnormal inputs): shifts of the 53-bit mantissa.
__device__ __noinline__ uint3 digits_wide_int(double a, int ex)
{
    uint32_t w[3];
    const unsigned long long b = (unsigned long long)__double_as_longlong(a);
    const uint32_t hi = (uint32_t)(b >> 32), lo = (uint32_t)b;
    const uint32_t negm = (uint32_t)((int32_t)hi >> 31);
    const int be = (int)((hi >> 20) & 0x7FFu);
    const uint32_t m1 = (hi & 0x000FFFFFu) | (be ? 0x00100000u : 0u), m0 = lo;
    const unsigned long long M = ((unsigned long long)m1 << 32) | m0;
    const int sh = (be ? be : 1) - 1075 + ex;                     // |a| 2^ex = M 2^sh, M < 2^53
    if (sh >= 0) {
        const int s = sh > 95 ? 95 : sh;
        const int ws = s >> 5, bs = s & 31;
        const uint32_t t0 = m0 << bs, t1 = __funnelshift_l(m0, m1, bs), t2 = __funnelshift_l(m1, 0u, bs);
        w[0] = ws == 0 ? t0 : 0u;
        w[1] = ws == 0 ? t1 : (ws == 1 ? t0 : 0u);
        w[2] = ws == 0 ? t2 : (ws == 1 ? t1 : t0);
    } else {
        const int r = -sh;
        const unsigned long long v = r < 64 ? (M >> r) : 0ull;    // dropping magnitude bits = toward zero
        w[0] = (uint32_t)v;
        w[1] = (uint32_t)(v >> 32);
        w[2] = 0u;
    }
    // two's complement over 96 bits, then + 2^95
    w[0] ^= negm; w[1] ^= negm; w[2] ^= negm;
    asm("add.cc.u32 %0, %0, %3;\n\taddc.cc.u32 %1, %1, 0;\n\taddc.u32 %2, %2, 0;"
        : "+r"(w[0]), "+r"(w[1]), "+r"(w[2]) : "r"(negm & 1u));
    w[2] ^= 0x80000000u;
    return make_uint3(w[0], w[1], w[2]);                          // by value: the caller's words stay in registers
}

// FP64 route (normal inputs): a' = th 2^32 + tl with th = trunc(a 2^(ex-32)) and tl = a 2^ex - th 2^32, both exact:
// th < 2^52 (|a'| < 2^84), and the remainder is a multiple of ulp(a 2^ex) below 2^32, so the FMA forms it without
// rounding.  th and tl carry the sign of a; their 96-bit two's-complement sum is assembled with one 64-bit add.
__device__ __forceinline__ void digits_wide(double a, int ex, uint32_t (&w)[3])
{
    const long long bits = __double_as_longlong(a);
    const int hi = (int)(bits >> 32);
    const int be = (hi >> 20) & 0x7FF;
    if (be == 0) {
        uint3 r = make_uint3(0u, 0u, 0x80000000u);
        if ((bits << 1) != 0) r = digits_wide_int(a, ex);
        w[0] = r.x; w[1] = r.y; w[2] = r.z;
        return;
    }
    const int ne = be + ex;                                       // biased exponent of a 2^ex
    const double x = __hiloint2double(hi + ex * 1048576, (int)bits);
    const double xh = __hiloint2double(hi + (ex - 32) * 1048576, (int)bits);
    const double hd = trunc(xh);                                  // |a 2^ex| >= 1 keeps a 2^(ex-32) a normal number
    const double rem = fma(hd, -4294967296.0, x);                 // exact
    long long th = __double2ll_rz(hd), tl = __double2ll_rz(rem);
    if (ne < 1023) { th = 0; tl = 0; }                            // |a 2^ex| < 1 truncates to 0
    const unsigned long long top = (unsigned long long)th << 32;
    const unsigned long long lo64 = top + (unsigned long long)tl;
    const int carry = lo64 < top ? 1 : 0;
    w[0] = (uint32_t)lo64;
    w[1] = (uint32_t)(lo64 >> 32);
    w[2] = ((uint32_t)((int)(th >> 32) + (int)(tl >> 63) + carry)) ^ 0x80000000u;
}

// The common case of both formats: when 2^ex is a normal double (|ex| <= 1022), a 2^ex is ONE exact FP64 multiply by the
// vector's scale -- also for subnormal a, and when the product falls below 1 (even into the subnormal range, where it may
// round) the truncation gives 0 as it must -- so trunc(a 2^ex) is a multiply and a conversion, with no exponent-field
// arithmetic.  Vectors whose exponent is outside that range (all entries below 2^-960 or so) take the routines above.
__device__ __forceinline__ bool scale_ok(int ex) { return ex >= -1022 && ex <= 1022; }
__device__ __forceinline__ double scale_of(int ex) { return __hiloint2double((ex + 1023) << 20, 0); }
__device__ __forceinline__ unsigned long long digits_narrow_scaled(double a, double scale)
{
    return (unsigned long long)__double2ll_rz(a * scale) ^ 0x8000000000000000ull;
}
__device__ __forceinline__ void digits_wide_scaled(double a, double scale, uint32_t (&w)[3])
{
    const double x = a * scale;                                   // exact (or below 1)
    const double hd = trunc(x * 2.3283064365386963e-10);          // th = trunc(a' / 2^32): exact, |.| < 2^52
    const double rem = fma(hd, -4294967296.0, x);                 // exact: a multiple of ulp(x) below 2^32 in magnitude
    const long long th = __double2ll_rz(hd), tl = __double2ll_rz(rem);
    const unsigned long long top = (unsigned long long)th << 32;
    const unsigned long long lo64 = top + (unsigned long long)tl;
    const int carry = lo64 < top ? 1 : 0;
    w[0] = (uint32_t)lo64;
    w[1] = (uint32_t)(lo64 >> 32);
    w[2] = ((uint32_t)((int)(th >> 32) + (int)(tl >> 63) + carry)) ^ 0x80000000u;
}
// the other vectors (rare, uniform for the warp): out of line
__device__ __noinline__ unsigned long long digits_narrow_slow(double a, int ex) { return digits_narrow(a, ex); }
__device__ __noinline__ uint3 digits_wide_slow(double a, int ex)
{
    uint32_t w[3];
    digits_wide(a, ex, w);
    return make_uint3(w[0], w[1], w[2]);
}

// ---------------------------------------------------------------------------------------------
// per-round tensor-core step and epilogue
// ---------------------------------------------------------------------------------------------
template <int WIDE>
struct ConvSmem {                                   // dynamic shared memory, 128-byte aligned base
    uint8_t tile[WIDE ? 2 : 1][CV_TILE_BYTES];      // K rows of digits 0 .. 7 (and 8 .. 11)
    uint8_t ones[CV_ONES_BYTES];
    uint8_t img[WIDE ? 6 : 2][CV_IMG_BYTES];        // narrow: weights, bias; wide: + high-digit weights, and all three for moduli 16 ..
    uint64_t mbar;
    uint32_t tmem_slot[2];
};

struct ConvCtx {
    uint32_t tile_row;          // shared address of this thread's 32-byte K row (first 16 bytes; +128 for the rest)
    uint32_t mbar;              // shared address of the MMA-done barrier
    uint32_t phase;
    uint32_t tmem;              // TMEM address of this thread's lane, column 0 (moduli 0 .. 15)
    uint32_t tmem_base;
    uint32_t tmem2, tmem2_base; // wide format: the 32-column accumulator of moduli 16 .. 19
    uint64_t adesc, bdesc, odesc, biasdesc;
    uint64_t ahdesc, bhdesc;    // wide format: K rows / weights of digits 8 .. 11
    uint64_t b2desc, bh2desc, bias2desc;
    uint32_t idesc, idesc2;     // idesc2 == 0: no second column group
};

__device__ __forceinline__ void sts128(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d)
{
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}

// all 128 K rows are in place: run the MMAs (digits x weights, ones x bias) and wait for the accumulator
template <int WIDE>
__device__ __forceinline__ void conv_mma(ConvCtx &cx)
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // generic-proxy stores -> tensor-core reads
    tc_fence_before();                                                // my tcgen05.ld of the previous round is done
    __syncthreads();
    if (threadIdx.x == 0) {
        tc_fence_after();
        tc_mma_i8(cx.tmem_base, cx.adesc, cx.bdesc, cx.idesc, 0u);
        if (WIDE) tc_mma_i8(cx.tmem_base, cx.ahdesc, cx.bhdesc, cx.idesc, 1u);
        tc_mma_i8(cx.tmem_base, cx.odesc, cx.biasdesc, cx.idesc, 1u);
        if (WIDE && cx.idesc2) {
            tc_mma_i8(cx.tmem2_base, cx.adesc, cx.b2desc, cx.idesc2, 0u);
            tc_mma_i8(cx.tmem2_base, cx.ahdesc, cx.bh2desc, cx.idesc2, 1u);
            tc_mma_i8(cx.tmem2_base, cx.odesc, cx.bias2desc, cx.idesc2, 1u);
        }
        tc_commit_a(cx.mbar);
    }
}
__device__ __forceinline__ void conv_wait(ConvCtx &cx)
{
    mbar_wait_a(cx.mbar, cx.phase);
    cx.phase ^= 1u;
    tc_fence_after();
}

// u = Y mod p for Y < 2^24 (exact: magic = floor(2^32 / p) + 1, Y (magic p - 2^32) < 2^32)
template <int L>
__device__ __forceinline__ uint32_t umod(uint32_t y)
{
    constexpr uint32_t p = modulus_of(L), magic = (uint32_t)(0x100000000ull / p) + 1u;
    return y - __umulhi(y, magic) * p;
}

// four residues of modulus L (accumulator values y0..y3 of the quad's four elements) -> one packed word of INT8
template <int L>
__device__ __forceinline__ uint32_t pack_quad(uint32_t y0, uint32_t y1, uint32_t y2, uint32_t y3)
{
    if constexpr (L == 0) {                                           // p = 256: the low bytes of a' (reading R5)
        return __byte_perm(__byte_perm(y0, y1, 0x0040), __byte_perm(y2, y3, 0x0040), 0x5410);
    } else {
        constexpr uint32_t half = (modulus_of(L) - 1) / 2, c = (128u - half) * 0x01010101u;
        const uint32_t u0 = umod<L>(y0), u1 = umod<L>(y1), u2 = umod<L>(y2), u3 = umod<L>(y3);
        const uint32_t w = __byte_perm(__byte_perm(u0, u1, 0x0040), __byte_perm(u2, u3, 0x0040), 0x5410);
        return (w + c) ^ 0x80808080u;                                 // per byte: u + 128 - half <= 255, then offset-128 -> INT8
    }
}

// narrow epilogue: accumulator column = 4 l + slot.  One LDTM per 8 moduli; moduli in groups of 4 with one uniform
// guard per group (and per-modulus guards in the last, partial group).
template <int L0>
__device__ __forceinline__ void store_group4(const uint32_t *v, int N, int8_t *dst, int64_t plane_stride)
{
    // v: 16 accumulator values (4 moduli x 4 slots) of moduli L0 .. L0 + 3
    if (L0 + 4 <= N) {
        *reinterpret_cast<uint32_t *>(dst + (int64_t)(L0 + 0) * plane_stride) = pack_quad<L0 + 0>(v[0], v[1], v[2], v[3]);
        *reinterpret_cast<uint32_t *>(dst + (int64_t)(L0 + 1) * plane_stride) = pack_quad<L0 + 1>(v[4], v[5], v[6], v[7]);
        *reinterpret_cast<uint32_t *>(dst + (int64_t)(L0 + 2) * plane_stride) = pack_quad<L0 + 2>(v[8], v[9], v[10], v[11]);
        *reinterpret_cast<uint32_t *>(dst + (int64_t)(L0 + 3) * plane_stride) = pack_quad<L0 + 3>(v[12], v[13], v[14], v[15]);
    } else {
        if (L0 + 0 < N) *reinterpret_cast<uint32_t *>(dst + (int64_t)(L0 + 0) * plane_stride) = pack_quad<L0 + 0>(v[0], v[1], v[2], v[3]);
        if (L0 + 1 < N) *reinterpret_cast<uint32_t *>(dst + (int64_t)(L0 + 1) * plane_stride) = pack_quad<L0 + 1>(v[4], v[5], v[6], v[7]);
        if (L0 + 2 < N) *reinterpret_cast<uint32_t *>(dst + (int64_t)(L0 + 2) * plane_stride) = pack_quad<L0 + 2>(v[8], v[9], v[10], v[11]);
    }
}

template <int WIDE>
__device__ __forceinline__ void conv_epilogue(const ConvCtx &cx, int N, int8_t *dst, int64_t plane_stride, bool ok)
{
    uint32_t v[32];
    tc_ld32(cx.tmem, v);
    if (ok) {
        store_group4<0>(v, N, dst, plane_stride);
        if (N > 4) store_group4<4>(v + 16, N, dst, plane_stride);
    }
    if (N > 8) {                                                      // uniform
        tc_ld32(cx.tmem + 32u, v);
        if (ok) {
            store_group4<8>(v, N, dst, plane_stride);
            if (N > 12) store_group4<12>(v + 16, N, dst, plane_stride);
        }
    }
    if (WIDE && N > 16) {                                             // uniform; second accumulator: moduli 16 .. 19
        tc_ld32(cx.tmem2, v);
        if (ok) store_group4<16>(v, N, dst, plane_stride);
    }
}

// one quad: digits -> K row(s) -> MMA -> residues of all N moduli -> 4-byte stores.  `overlap()` runs between the MMA
// issue and the wait for its result (the callers put the loads of their next work item there).
template <int WIDE, typename F>
__device__ __forceinline__ void convert_quad(ConvCtx &cx, const double (&a)[4], int ex, int N, int8_t *dst,
                                             int64_t plane_stride, bool ok, F overlap)
{
    const double scale = scale_of(ex);
    if (!WIDE) {
        unsigned long long d[4];
        if (scale_ok(ex)) {                                                   // uniform for the warp
#pragma unroll
            for (int u = 0; u < 4; u++) d[u] = digits_narrow_scaled(a[u], scale);
        } else {
#pragma unroll
            for (int u = 0; u < 4; u++) d[u] = digits_narrow_slow(a[u], ex);
        }
        sts128(cx.tile_row, (uint32_t)d[0], (uint32_t)(d[0] >> 32), (uint32_t)d[1], (uint32_t)(d[1] >> 32));
        sts128(cx.tile_row + 128u, (uint32_t)d[2], (uint32_t)(d[2] >> 32), (uint32_t)d[3], (uint32_t)(d[3] >> 32));
    } else {
        uint32_t w0[3], w1[3], w2[3], w3[3];
        if (scale_ok(ex)) {                                                   // uniform for the warp
            digits_wide_scaled(a[0], scale, w0);
            digits_wide_scaled(a[1], scale, w1);
            digits_wide_scaled(a[2], scale, w2);
            digits_wide_scaled(a[3], scale, w3);
        } else {
            uint3 r = digits_wide_slow(a[0], ex); w0[0] = r.x; w0[1] = r.y; w0[2] = r.z;
            r = digits_wide_slow(a[1], ex); w1[0] = r.x; w1[1] = r.y; w1[2] = r.z;
            r = digits_wide_slow(a[2], ex); w2[0] = r.x; w2[1] = r.y; w2[2] = r.z;
            r = digits_wide_slow(a[3], ex); w3[0] = r.x; w3[1] = r.y; w3[2] = r.z;
        }
        sts128(cx.tile_row, w0[0], w0[1], w1[0], w1[1]);
        sts128(cx.tile_row + 128u, w2[0], w2[1], w3[0], w3[1]);
        sts128(cx.tile_row + CV_TILE_BYTES, w0[2], 0u, w1[2], 0u);             // digits 8 .. 11 (12 .. 15 are zero)
        sts128(cx.tile_row + CV_TILE_BYTES + 128u, w2[2], 0u, w3[2], 0u);
    }
    conv_mma<WIDE>(cx);
    overlap();
    conv_wait(cx);
    conv_epilogue<WIDE>(cx, N, dst, plane_stride, ok);
}

// CTA prologue: operand images, barrier, tensor memory
template <int WIDE>
__device__ __forceinline__ void conv_setup(ConvSmem<WIDE> *S, ConvCtx &cx, int N)
{
    const int tid = threadIdx.x;
    // images: narrow {weights, bias}; wide {weights lo, weights hi, bias} for moduli 0 .. 15 and the same for 16 .. 19
    for (int t = tid; t < CV_IMG_BYTES / 16; t += CV_THREADS) {
        if (!WIDE) {
            reinterpret_cast<uint4 *>(S->img[0])[t] = reinterpret_cast<const uint4 *>(g_conv_img[0][0])[t];
            reinterpret_cast<uint4 *>(S->img[1])[t] = reinterpret_cast<const uint4 *>(g_conv_img[0][2])[t];
        } else {
#pragma unroll
            for (int g = 0; g < 2; g++) {
                reinterpret_cast<uint4 *>(S->img[3 * g + 0])[t] = reinterpret_cast<const uint4 *>(g_conv_img[g][0])[t];
                reinterpret_cast<uint4 *>(S->img[3 * g + 1])[t] = reinterpret_cast<const uint4 *>(g_conv_img[g][1])[t];
                reinterpret_cast<uint4 *>(S->img[3 * g + 2])[t] = reinterpret_cast<const uint4 *>(g_conv_img[g][3])[t];
            }
        }
    }
    if (tid < CV_ONES_BYTES / 16)                                     // K byte 0 of every row = 1: first byte of the 8 core rows of K chunk 0
        reinterpret_cast<uint4 *>(S->ones)[tid] = make_uint4(tid < 8 ? 1u : 0u, 0u, 0u, 0u);
    if (tid == 0) {
        mbar_init(&S->mbar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    const bool second = WIDE && N > 16;
    if (tid < 32) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&S->tmem_slot[0])), "n"(CV_TMEM_COLS) : "memory");
        if (second)
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 32;" ::"r"(smem_u32(&S->tmem_slot[1])) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t lane_off = (uint32_t)(tid & ~31) << 16;            // lane quarter of this warp
    cx.tmem_base = S->tmem_slot[0];
    cx.tmem = cx.tmem_base + lane_off;
    cx.tmem2_base = second ? S->tmem_slot[1] : 0u;
    cx.tmem2 = cx.tmem2_base + lane_off;
    cx.tile_row = smem_u32(S->tile[0]) + (uint32_t)tile_off(tid, 0);
    cx.mbar = smem_u32(&S->mbar);
    cx.phase = 0;
    cx.adesc = kmajor_desc(smem_u32(S->tile[0]), 256u);
    cx.odesc = kmajor_desc(smem_u32(S->ones), 0u);                    // every 8-row group reads the same 256 bytes
    cx.bdesc = kmajor_desc(smem_u32(S->img[0]), 256u);
    if (!WIDE) {
        cx.biasdesc = kmajor_desc(smem_u32(S->img[1]), 256u);
        cx.ahdesc = cx.bhdesc = cx.b2desc = cx.bh2desc = cx.bias2desc = 0;
    } else {
        cx.ahdesc = kmajor_desc(smem_u32(S->tile[WIDE ? 1 : 0]), 256u);
        cx.bhdesc = kmajor_desc(smem_u32(S->img[1]), 256u);
        cx.biasdesc = kmajor_desc(smem_u32(S->img[2]), 256u);
        cx.b2desc = kmajor_desc(smem_u32(S->img[WIDE ? 3 : 0]), 256u);
        cx.bh2desc = kmajor_desc(smem_u32(S->img[WIDE ? 4 : 0]), 256u);
        cx.bias2desc = kmajor_desc(smem_u32(S->img[WIDE ? 5 : 0]), 256u);
    }
    // accumulator columns in use: 4 per modulus, rounded up to the MMA's N granule of 16; moduli 16 .. 19 in the second group
    const int n1 = N < 16 ? N : 16;
    const uint32_t nmma = (uint32_t)((4 * n1 + 15) & ~15);
    // kind::i8: D = S32, A = B = unsigned 8 bit, both K-major, M = 128
    cx.idesc = (2u << 4) | ((nmma >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
    cx.idesc2 = second ? ((2u << 4) | ((16u >> 3) << 17) | ((uint32_t)(128 >> 4) << 24)) : 0u;
}

__device__ __forceinline__ void conv_teardown(const ConvCtx &cx)
{
    tc_fence_before();
    __syncthreads();
    if (threadIdx.x < 32) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(cx.tmem_base), "n"(CV_TMEM_COLS) : "memory");
        if (cx.idesc2) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 32;" ::"r"(cx.tmem2_base) : "memory");
    }
}

template <int WIDE>
__device__ __forceinline__ ConvSmem<WIDE> *conv_smem(uint8_t *raw)
{
    return reinterpret_cast<ConvSmem<WIDE> *>((reinterpret_cast<uintptr_t>(raw) + 127) & ~(uintptr_t)127);   // no swizzle: 16 B would do
}

// four consecutive elements of a contiguous vector as doubles: two 16-byte loads (FP64) or one (FP32)
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
template <typename T>
__device__ __forceinline__ void load_quad(const T *vec, int64_t h, int64_t k, bool vec_ok, double (&a)[4])
{
    if (vec_ok && h + 3 < k) ld4(vec + h, a);
    else {
#pragma unroll
        for (int u = 0; u < 4; u++) a[u] = (h + u < k) ? (double)__ldg(vec + h + u) : 0.0;
    }
}

// ---------------------------------------------------------------------------------------------
// contiguous vectors: vector j is X[h + j ldx].  Work item = (vector, chunk of 512 h), persistent CTAs.
// ---------------------------------------------------------------------------------------------
template <int WIDE, typename T>
__global__ void __launch_bounds__(CV_THREADS, WIDE ? 5 : 8)
k2_tc_cols(int N, int64_t rows, int64_t k, const T *__restrict__ X, int64_t ldx, const int32_t *__restrict__ ex,
           int8_t *__restrict__ planes, int64_t kp)
{
    extern __shared__ uint8_t smem_raw[];
    ConvSmem<WIDE> *S = conv_smem<WIDE>(smem_raw);
    ConvCtx cx;
    conv_setup<WIDE>(S, cx, N);
    pdl_launch_dependents();                         // after the tensor-memory allocation of conv_setup (oz2_common.cuh)
    pdl_wait();                                      // the exponents come from the scaling kernels
    const int tid = threadIdx.x;
    const int chunks = (int)((kp + CV_CHUNK_H - 1) / CV_CHUNK_H);      // k <= 2^22: fits 32 bits
    const int64_t items = rows * chunks;
    const int64_t plane_stride = rows * kp;
    const int k32 = (int)k, kp32 = (int)kp;
    // items are dealt round-robin (item = blockIdx.x + t gridDim.x): at any time the CTAs work on neighbouring chunks, so
    // that reads and the N write streams stay sequential across the chip.  (j, c) advance without a division.
    const int step_j = (int)(gridDim.x / (unsigned)chunks), step_c = (int)(gridDim.x - (unsigned)step_j * (unsigned)chunks);
    int j = (int)(blockIdx.x / (unsigned)chunks), c = (int)(blockIdx.x - (unsigned)j * (unsigned)chunks);
    double a[4] = { 0.0, 0.0, 0.0, 0.0 };
    int e = 0;
    auto fetch = [&](int jj, int cc) {
        const T *vec = X + (int64_t)jj * ldx;
        const int h = cc * CV_CHUNK_H + 4 * tid;
        if (((((uintptr_t)vec) & 15) == 0) && h + 3 < k32) ld4(vec + h, a);
        else {
#pragma unroll
            for (int u = 0; u < 4; u++) a[u] = (h + u < k32) ? (double)__ldg(vec + h + u) : 0.0;
        }
        e = __ldg(ex + jj);
    };
    if ((int64_t)blockIdx.x < items) fetch(j, c);
    for (int64_t item = blockIdx.x; item < items; item += gridDim.x) {
        const double cur[4] = { a[0], a[1], a[2], a[3] };
        const int ecur = e;
        const int h = c * CV_CHUNK_H + 4 * tid;
        int8_t *dst = planes + (int64_t)j * kp + h;
        const bool ok = h < kp32;
        c += step_c; j += step_j;
        if (c >= chunks) { c -= chunks; j++; }
        // next item: its loads are in flight while this one runs through the tensor core and the epilogue
        convert_quad<WIDE>(cx, cur, ecur, N, dst, plane_stride, ok, [&] { if (item + gridDim.x < items) fetch(j, c); });
    }
    conv_teardown(cx);
}

// ---------------------------------------------------------------------------------------------
// strided vectors: vector i is X[i + h ldx] (rows of a column-major matrix).  Work item = block of 16 vectors x 128 h,
// brought into shared memory by cp.async (128-byte coalesced reads along the rows, transposed on the way in); four
// rounds of 4 vectors x 128 h per block (a warp = one vector, 128 contiguous bytes per store).  The copy of the next
// block is issued as soon as the last round has read the buffer, so it overlaps that round's MMA and epilogue.
// ---------------------------------------------------------------------------------------------
constexpr int ST_ROWS = 16, ST_H = 128;
template <typename T>
struct StageRow { static constexpr int PITCH = ST_H + 16 / (int)sizeof(T); };      // 16-byte aligned rows, odd in 16-byte units

__device__ __forceinline__ void cp_async_zfill(uint32_t dst, const void *src, bool valid, int bytes)
{
    // copies `bytes` (4 or 8) or, if !valid, writes zeros (src-size 0); src must be a valid address either way
    if (bytes == 8)
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(dst), "l"(src), "r"(valid ? 8 : 0) : "memory");
    else
        asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(dst), "l"(src), "r"(valid ? 4 : 0) : "memory");
}

template <int WIDE, typename T>
__global__ void __launch_bounds__(CV_THREADS, WIDE ? 5 : 8)
k2_tc_rows(int N, int64_t rows, int64_t k, const T *__restrict__ X, int64_t ldx, const int32_t *__restrict__ ex,
           int8_t *__restrict__ planes, int64_t kp)
{
    extern __shared__ uint8_t smem_raw[];
    ConvSmem<WIDE> *S = conv_smem<WIDE>(smem_raw);
    constexpr int PITCH = StageRow<T>::PITCH;
    T *stage = reinterpret_cast<T *>(S + 1);
    ConvCtx cx;
    conv_setup<WIDE>(S, cx, N);
    pdl_launch_dependents();                         // after the tensor-memory allocation of conv_setup (oz2_common.cuh)
    pdl_wait();                                      // the exponents come from the scaling kernels
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nib = (int)((rows + ST_ROWS - 1) / ST_ROWS), nhb = (int)(kp / ST_H);
    const int64_t items = (int64_t)nib * nhb;
    const int64_t plane_stride = rows * kp;
    const int k32 = (int)k;
    // item = ib + nib hb (row blocks fastest: concurrent CTAs read whole columns), walked with stride gridDim.x
    const int step_hb = (int)(gridDim.x / (unsigned)nib), step_ib = (int)(gridDim.x - (unsigned)step_hb * (unsigned)nib);
    int hb = (int)(blockIdx.x / (unsigned)nib), ib = (int)(blockIdx.x - (unsigned)hb * (unsigned)nib);
    // copy pattern: thread = (row r = tid % 16, h = tid / 16 + 8 s), s = 0 .. 15
    const int r = tid & 15, hs = tid >> 4;
    const uint32_t stage_s = smem_u32(stage) + (uint32_t)((r * PITCH + hs) * sizeof(T));
    auto issue = [&](int ibn, int hbn) {
        const int64_t i = (int64_t)ibn * ST_ROWS + r;
        const int h0 = hbn * ST_H + hs;
        const bool rok = i < rows;
        const T *srcp = X + (rok ? i : 0) + (int64_t)h0 * ldx;
#pragma unroll
        for (int s = 0; s < ST_H / 8; s++) {
            const bool v = rok && h0 + 8 * s < k32;
            cp_async_zfill(stage_s + (uint32_t)(8 * s * sizeof(T)), v ? srcp + (int64_t)(8 * s) * ldx : X, v, (int)sizeof(T));
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    if ((int64_t)blockIdx.x < items) issue(ib, hb);
    for (int64_t item = blockIdx.x; item < items; item += gridDim.x) {
        const int ibc = ib, hbc = hb;
        ib += step_ib; hb += step_hb;
        if (ib >= nib) { ib -= nib; hb++; }
        const bool more = item + gridDim.x < items;
        // exponents of this thread's four vectors (one per round)
        int e4[4];
#pragma unroll
        for (int rr = 0; rr < 4; rr++) {
            const int64_t i = (int64_t)ibc * ST_ROWS + 4 * rr + warp;
            e4[rr] = i < rows ? __ldg(ex + i) : 0;
        }
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();                                                   // every thread's copies of this block have landed
#pragma unroll
        for (int rr = 0; rr < ST_ROWS / 4; rr++) {
            const int rl = 4 * rr + warp;
            const int64_t i = (int64_t)ibc * ST_ROWS + rl;
            const bool ok = i < rows;
            double a[4];
            if constexpr (sizeof(T) == 8) {
                const double2 lo = *reinterpret_cast<const double2 *>(&stage[rl * PITCH + 4 * lane]);
                const double2 hi = *reinterpret_cast<const double2 *>(&stage[rl * PITCH + 4 * lane + 2]);
                a[0] = lo.x; a[1] = lo.y; a[2] = hi.x; a[3] = hi.y;
            } else {
                const float4 q = *reinterpret_cast<const float4 *>(&stage[rl * PITCH + 4 * lane]);
                a[0] = (double)q.x; a[1] = (double)q.y; a[2] = (double)q.z; a[3] = (double)q.w;
            }
            int8_t *dst = planes + i * kp + hbc * ST_H + 4 * lane;
            // after the barrier inside the last round every thread has read the buffer: refill it for the next block
            convert_quad<WIDE>(cx, a, e4[rr], N, dst, plane_stride, ok, [&] { if (rr == ST_ROWS / 4 - 1 && more) issue(ib, hb); });
        }
    }
    conv_teardown(cx);
}

// ---------------------------------------------------------------------------------------------
// accurate mode: Abar / Bbar = ceil(|a| 2^(5-E)) in [0, 64], one INT8 plane, CUDA cores only
// ---------------------------------------------------------------------------------------------
__device__ __noinline__ uint32_t ceil_scaled(double a, int E)
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
    const int g = E < -4096 ? 4096 : 5 - E;           // the all-zero marker takes the integer route (which returns zeros)
    if (g >= -1022 && g <= 1023) {
        // |a| 2^g is an exact FP64 multiply while it stays normal; if it underflows, rounding up keeps it in (0, 1) and the
        // ceiling is 1 as it must be; 0 stays 0.  (E of an all-zero vector is a marker far outside this range.)
        const double scale = __hiloint2double((g + 1023) << 20, 0);
#pragma unroll
        for (int u = 0; u < 4; u++) o |= (uint32_t)__double2int_ru(__dmul_ru(fabs(a[u]), scale)) << (8 * u);
    } else {
#pragma unroll
        for (int u = 0; u < 4; u++) o |= ceil_scaled(a[u], E) << (8 * u);
    }
    *reinterpret_cast<uint32_t *>(dst) = o;
}

constexpr int BAR_TI = 32, BAR_TH = 128, BAR_SROW = BAR_TH + 2, BAR_THREADS = 256;

template <typename T>
__global__ void __launch_bounds__(BAR_THREADS)
k2_bar_rows(int64_t m, int64_t k, const T *__restrict__ A, int64_t lda, const int32_t *__restrict__ E, int8_t *__restrict__ plane,
            int64_t kp)
{
    __shared__ __align__(16) double tile[BAR_TI * BAR_SROW];
    pdl_launch_dependents();
    pdl_wait();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t i0 = (int64_t)blockIdx.x * BAR_TI, h0 = (int64_t)blockIdx.y * BAR_TH;
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
        for (int s = 0; s < 16; s++) tile[lane * BAR_SROW + warp + 8 * s] = v[s];
    }
    __syncthreads();
#pragma unroll 1
    for (int rr = 0; rr < BAR_TI / 8; rr++) {
        const int il = warp * (BAR_TI / 8) + rr;
        const int64_t i = i0 + il;
        if (i >= m) break;
        const double2 lo = *reinterpret_cast<const double2 *>(&tile[il * BAR_SROW + 4 * lane]);
        const double2 hi = *reinterpret_cast<const double2 *>(&tile[il * BAR_SROW + 4 * lane + 2]);
        const double a[4] = { lo.x, lo.y, hi.x, hi.y };
        quad_bar(a, __ldg(E + i), plane + i * kp + h0 + 4 * lane);
    }
}

template <typename T>
__global__ void __launch_bounds__(BAR_THREADS)
k2_bar_cols(int64_t n, int64_t k, const T *__restrict__ B, int64_t ldb, const int32_t *__restrict__ E, int8_t *__restrict__ plane,
            int64_t kp)
{
    pdl_launch_dependents();
    pdl_wait();
    const int64_t quads = kp / 4;
    const int64_t t = (int64_t)blockIdx.x * BAR_THREADS + threadIdx.x;
    if (t >= n * quads) return;
    const int64_t j = t / quads, h = (t - j * quads) * 4;
    const T *col = B + j * ldb;
    double a[4];
    load_quad(col, h, k, (((uintptr_t)col) & 15) == 0, a);
    quad_bar(a, __ldg(E + j), plane + j * kp + h);
}

template <int WIDE, typename T>
constexpr size_t rows_smem() { return sizeof(ConvSmem<WIDE>) + 128 + (size_t)ST_ROWS * StageRow<T>::PITCH * sizeof(T); }
template <int WIDE>
constexpr size_t cols_smem() { return sizeof(ConvSmem<WIDE>) + 128; }

template <typename T>
int launch_convert_t(int op, int N, int wide, int64_t rows, int64_t k, const T *X, int64_t ldx, const int32_t *ex,
                     int8_t *planes, int64_t kp, cudaStream_t st)
{
    if (N == 0) {                                     // accurate mode's single plane
        if (op == 0) {
            dim3 grid((unsigned)((rows + BAR_TI - 1) / BAR_TI), (unsigned)(kp / BAR_TH));
            OZ2_CUDA_TRY(oz2_launch(k2_bar_rows<T>, grid, dim3(BAR_THREADS), 0, st, rows, k, X, ldx, ex, planes, kp));
        } else {
            const int64_t total = rows * (kp / 4);
            OZ2_CUDA_TRY(oz2_launch(k2_bar_cols<T>, dim3((unsigned)((total + BAR_THREADS - 1) / BAR_THREADS)), dim3(BAR_THREADS), 0, st, rows, k, X, ldx, ex, planes, kp));
        }
    } else {
        const int per_sm = wide ? 5 : 8;              // tensor memory: 64 (+ 32) columns per CTA
        if (op == 0) {
            const int64_t items = ((rows + ST_ROWS - 1) / ST_ROWS) * (kp / ST_H);
            int64_t grid = (int64_t)oz2_num_sms() * per_sm;
            if (grid > items) grid = items;
            if (wide) OZ2_CUDA_TRY(oz2_launch(k2_tc_rows<1, T>, dim3((unsigned)grid), dim3(CV_THREADS), rows_smem<1, T>(), st, N, rows, k, X, ldx, ex, planes, kp));
            else OZ2_CUDA_TRY(oz2_launch(k2_tc_rows<0, T>, dim3((unsigned)grid), dim3(CV_THREADS), rows_smem<0, T>(), st, N, rows, k, X, ldx, ex, planes, kp));
        } else {
            const int64_t items = rows * ((kp + CV_CHUNK_H - 1) / CV_CHUNK_H);
            int64_t grid = (int64_t)oz2_num_sms() * per_sm;
            if (grid > items) grid = items;
            if (wide) OZ2_CUDA_TRY(oz2_launch(k2_tc_cols<1, T>, dim3((unsigned)grid), dim3(CV_THREADS), cols_smem<1>(), st, N, rows, k, X, ldx, ex, planes, kp));
            else OZ2_CUDA_TRY(oz2_launch(k2_tc_cols<0, T>, dim3((unsigned)grid), dim3(CV_THREADS), cols_smem<0>(), st, N, rows, k, X, ldx, ex, planes, kp));
        }
    }
    oz2_count_launches(1);
    OZ2_CUDA_TRY(cudaGetLastError());
    return 0;
}

} // namespace

int oz2_convert_upload_tables(const Oz2HostTables &t)
{
    static uint8_t img[2][4][CV_IMG_BYTES];
    memset(img, 0, sizeof(img));
    for (int l = 0; l < OZ2_MAX_MODULI; l++) {
        const uint32_t p = t.mod[l].p, half = (p - 1) / 2;
        const int g = l / 16;
        uint32_t two = 1 % p, bias[2] = { 0u, 0u };                  // 2^b mod p; bias = half - 2^topbit mod p: Y ~ a' + half (mod p)
        for (int b = 0; b <= 95; b++) {
            if (b == 63) bias[0] = (half + p - two) % p;
            if (b == 95) bias[1] = (half + p - two) % p;
            two = (two * 2u) % p;
        }
        if (l == 0) bias[0] = bias[1] = 0u;                           // p = 256 keeps the low byte of a'
        for (int s = 0; s < 4; s++) {
            const int col = (l % 16) * 4 + s;
            for (int i = 0; i < 12; i++) {
                const uint32_t w = (t.mod[l].wb[i / 4] >> (8 * (i % 4))) & 0xFFu;          // 256^i mod p
                if (i < 8) img[g][0][tile_off(col, 8 * s + i)] = (uint8_t)w;
                else img[g][1][tile_off(col, 8 * s + i - 8)] = (uint8_t)w;
            }
            img[g][2][tile_off(col, 0)] = (uint8_t)bias[0];
            img[g][3][tile_off(col, 0)] = (uint8_t)bias[1];
        }
    }
    OZ2_CUDA_TRY(cudaMemcpyToSymbol(g_conv_img, img, sizeof(img)));
    OZ2_CUDA_TRY(cudaFuncSetAttribute(k2_tc_rows<0, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rows_smem<0, double>()));
    OZ2_CUDA_TRY(cudaFuncSetAttribute(k2_tc_rows<1, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rows_smem<1, double>()));
    OZ2_CUDA_TRY(cudaFuncSetAttribute(k2_tc_rows<0, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rows_smem<0, float>()));
    OZ2_CUDA_TRY(cudaFuncSetAttribute(k2_tc_rows<1, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rows_smem<1, float>()));
    return 0;
}

// op 0: strided vectors (rows of a column-major matrix), op 1: contiguous vectors (its columns).  N >= 1: residue
// planes [N][rows][kp] with exponents `ex`; wide != 0 when |a'| may exceed 63 bits.  N == 0: the single plane
// ceil(mu' |.|) of accurate mode; `ex` then holds E = floor(log2 max |.|) per vector.
// f32 != 0: X is FP32 (SGEMM variant), promoted exactly on load.
int oz2_launch_convert(int op, int N, int wide, int f32, int64_t rows, int64_t k, const void *X, int64_t ldx,
                       const int32_t *ex, int8_t *planes, int64_t kp, cudaStream_t st)
{
    if (rows <= 0) return 0;
    if (f32) return launch_convert_t<float>(op, N, wide, rows, k, static_cast<const float *>(X), ldx, ex, planes, kp, st);
    return launch_convert_t<double>(op, N, wide, rows, k, static_cast<const double *>(X), ldx, ex, planes, kp, st);
}
