// oz2_convert.cu -- S2: A' = trunc(diag(mu) A), B' = trunc(B diag(nu)) (Step 2) and the symmetric
// INT8 residues rmod(., p_l) for all N moduli in ONE pass over A and B.
//
// The scaled integers (up to 84 bits, never materialised in memory) live in registers as NB 32-bit words
// (magnitude) plus a sign.  The residue modulo an odd p is taken from the base-256 digits:
//     |a'| = sum_i d_i 256^i   =>   |a'| mod p = (sum_i d_i (256^i mod p)) mod p,
// i.e. NB dp4a instructions against packed byte weights, one mulhi-based exact reduction that lands directly
// in the symmetric range, then the sign.  p = 256 is the low byte in two's complement (reading R5).
//
// Layout written: planes[l][row][kp], k fastest (K-major for the tensor-core GEMM), kp = round_up(k, 128),
// padding zero filled.  A is column-major, so the A path maps one thread to one row (coalesced loads along
// the rows of a column) and stores 16 bytes per modulus; B's columns are already K-major: a warp walks 512
// consecutive h of one column with fully coalesced 4-byte stores per modulus.
#include "oz2_common.cuh"

namespace {

__constant__ Oz2ModTab c_mod[OZ2_MAX_MODULI];

// magnitude words of trunc(|a| 2^ex) and the sign of a
template <int NB>
__device__ __forceinline__ void scaled_words(double a, int ex, uint32_t (&w)[NB], uint32_t &neg)
{
    unsigned long long b = (unsigned long long)__double_as_longlong(a);
    neg = (uint32_t)(b >> 63);
    int be = (int)((b >> 52) & 0x7FF);
    unsigned long long mant = b & 0x000FFFFFFFFFFFFFull;
    unsigned long long M = be ? (mant | 0x0010000000000000ull) : mant;
    int sh = (be ? be : 1) - 1075 + ex;          // |a| 2^ex = M 2^sh
    uint32_t m0 = (uint32_t)M, m1 = (uint32_t)(M >> 32);
    if (sh >= 0 && be != 0) {
        // normal number: left shift by 0..31 (the row's largest element has 53 + sh <= 84 bits, every other
        // |a| is below twice the largest)
        w[0] = m0 << sh;
        w[1] = __funnelshift_l(m0, m1, sh);
        if (NB == 3) w[2] = __funnelshift_l(m1, 0u, sh);
    } else if (sh >= 0) {
        // subnormal number with a short mantissa: the shift can reach 83
        unsigned long long lo = sh < 64 ? (M << sh) : 0ull;
        w[0] = (uint32_t)lo;
        w[1] = (uint32_t)(lo >> 32);
        if (NB == 3) w[2] = sh == 0 ? 0u : (sh < 64 ? (uint32_t)(M >> (64 - sh)) : (uint32_t)(M << (sh - 64)));
    } else {
        int r = -sh;
        unsigned long long v = r < 64 ? (M >> r) : 0ull;      // dropping magnitude bits = toward zero
        w[0] = (uint32_t)v;
        w[1] = (uint32_t)(v >> 32);
        if (NB == 3) w[2] = 0u;
    }
}

// symmetric residue of +-V modulo the odd modulus described by t
template <int NB>
__device__ __forceinline__ int residue_odd(const uint32_t (&w)[NB], uint32_t neg, const Oz2ModTab &t)
{
    uint32_t x = __dp4a(w[0], t.wb[0], 0u);
    x = __dp4a(w[1], t.wb[1], x);
    if (NB == 3) x = __dp4a(w[2], t.wb[2], x);
    uint32_t q = __umulhi(x + t.half, t.magic);              // floor((x + h) / p) = round(x / p), exact (x < 2^24)
    int r = (int)x - (int)(q * t.p);                         // in [-h, h], congruent to |a'|
    return neg ? -r : r;
}

template <int NB>
__device__ __forceinline__ int residue_256(const uint32_t (&w)[NB], uint32_t neg)
{
    int b0 = (int)(w[0] & 0xFFu);
    return (neg ? -b0 : b0) & 0xFF;                          // two's-complement low byte of a'
}

// ---------------------------------------------------------------------------------------------
// A path: thread = row i, 16 consecutive h per iteration
// ---------------------------------------------------------------------------------------------
template <int NB>
__global__ void __launch_bounds__(128)
k2_rows(int N, int64_t m, int64_t k, const double *__restrict__ A, int64_t lda, const int32_t *__restrict__ e,
        int8_t *__restrict__ planes, int64_t kp)
{
    int64_t i = (int64_t)blockIdx.x * 128 + threadIdx.x;
    if (i >= m) return;
    const int ex = e[i];
    const int64_t plane_stride = m * kp;
    const int64_t chunk = oz2_round_up((kp / 16 + gridDim.y - 1) / gridDim.y, 8) * 16;   // multiple of 128 bytes
    const int64_t hbeg = (int64_t)blockIdx.y * chunk, hend = hbeg + chunk < kp ? hbeg + chunk : kp;
    for (int64_t h0 = hbeg; h0 < hend; h0 += 16) {
        uint32_t w[16][NB];
        uint32_t negmask = 0;
#pragma unroll
        for (int u = 0; u < 16; u++) {
            int64_t h = h0 + u;
            double a = h < k ? __ldg(A + i + h * lda) : 0.0;
            uint32_t neg;
            scaled_words<NB>(a, ex, w[u], neg);
            negmask |= neg << u;
        }
        int8_t *dst = planes + i * kp + h0;
        {   // p = 256
            uint32_t o[4] = { 0, 0, 0, 0 };
#pragma unroll
            for (int u = 0; u < 16; u++) o[u >> 2] |= (uint32_t)residue_256<NB>(w[u], (negmask >> u) & 1u) << (8 * (u & 3));
            *reinterpret_cast<uint4 *>(dst) = make_uint4(o[0], o[1], o[2], o[3]);
        }
#pragma unroll 1
        for (int l = 1; l < N; l++) {
            const Oz2ModTab t = c_mod[l];
            uint32_t o[4] = { 0, 0, 0, 0 };
#pragma unroll
            for (int u = 0; u < 16; u++)
                o[u >> 2] |= ((uint32_t)residue_odd<NB>(w[u], (negmask >> u) & 1u, t) & 0xFFu) << (8 * (u & 3));
            *reinterpret_cast<uint4 *>(dst + l * plane_stride) = make_uint4(o[0], o[1], o[2], o[3]);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// B path: warp = 512 consecutive h of column j; lane holds h = c*512 + 128 t + 4 lane + {0..3}, t = 0..3
// ---------------------------------------------------------------------------------------------
template <int NB>
__global__ void __launch_bounds__(128)
k2_cols(int N, int64_t n, int64_t k, const double *__restrict__ B, int64_t ldb, const int32_t *__restrict__ f,
        int8_t *__restrict__ planes, int64_t kp)
{
    const int lane = threadIdx.x & 31;
    const int64_t chunks = (kp + 511) / 512;
    const int64_t items = n * chunks;
    const int64_t plane_stride = n * kp;
    for (int64_t it = (int64_t)blockIdx.x * 4 + (threadIdx.x >> 5); it < items; it += (int64_t)gridDim.x * 4) {
        const int64_t j = it / chunks, c = it - j * chunks;
        const double *col = B + j * ldb;
        const int ex = f[j];
        const bool vec = ((((uintptr_t)col) & 15) == 0);
        uint32_t w[16][NB];
        uint32_t negmask = 0;
#pragma unroll
        for (int t = 0; t < 4; t++) {
            int64_t h = c * 512 + 128 * t + 4 * lane;
            double a[4];
            if (vec && h + 3 < k) {
                double2 v0 = __ldg(reinterpret_cast<const double2 *>(col + h));
                double2 v1 = __ldg(reinterpret_cast<const double2 *>(col + h + 2));
                a[0] = v0.x; a[1] = v0.y; a[2] = v1.x; a[3] = v1.y;
            } else {
#pragma unroll
                for (int u = 0; u < 4; u++) a[u] = (h + u < k) ? __ldg(col + h + u) : 0.0;
            }
#pragma unroll
            for (int u = 0; u < 4; u++) {
                uint32_t neg;
                scaled_words<NB>(a[u], ex, w[4 * t + u], neg);
                negmask |= neg << (4 * t + u);
            }
        }
        int8_t *dst = planes + j * kp + c * 512 + 4 * lane;
#pragma unroll 1
        for (int l = 0; l < N; l++) {
            const Oz2ModTab tb = c_mod[l];
#pragma unroll
            for (int t = 0; t < 4; t++) {
                uint32_t o = 0;
#pragma unroll
                for (int u = 0; u < 4; u++) {
                    int r = l == 0 ? residue_256<NB>(w[4 * t + u], (negmask >> (4 * t + u)) & 1u)
                                   : residue_odd<NB>(w[4 * t + u], (negmask >> (4 * t + u)) & 1u, tb);
                    o |= ((uint32_t)r & 0xFFu) << (8 * u);
                }
                if (c * 512 + 128 * t + 4 * lane < kp)
                    *reinterpret_cast<uint32_t *>(dst + l * plane_stride + 128 * t) = o;
            }
        }
    }
}

} // namespace

int oz2_convert_upload_tables(const Oz2HostTables &t)
{
    OZ2_CUDA_TRY(cudaMemcpyToSymbol(c_mod, t.mod, sizeof(t.mod)));
    return 0;
}

int oz2_launch_convert(int op, int N, int wide, int64_t rows, int64_t k, const double *X, int64_t ldx,
                       const int32_t *ex, int8_t *planes, int64_t kp, cudaStream_t st)
{
    if (rows <= 0) return 0;
    if (op == 0) {
        int64_t bx = (rows + 127) / 128;
        int64_t gy = (148 * 12 + bx - 1) / bx;
        int64_t chunks = kp / 16;
        if (gy > chunks) gy = chunks;
        if (gy > 65535) gy = 65535;
        if (gy < 1) gy = 1;
        dim3 grid((unsigned)bx, (unsigned)gy);
        if (wide) k2_rows<3><<<grid, 128, 0, st>>>(N, rows, k, X, ldx, ex, planes, kp);
        else k2_rows<2><<<grid, 128, 0, st>>>(N, rows, k, X, ldx, ex, planes, kp);
    } else {
        int64_t items = rows * ((kp + 511) / 512);
        int64_t gx = (items + 3) / 4;
        if (gx > 148 * 32) gx = 148 * 32;
        if (wide) k2_cols<3><<<(unsigned)gx, 128, 0, st>>>(N, rows, k, X, ldx, ex, planes, kp);
        else k2_cols<2><<<(unsigned)gx, 128, 0, st>>>(N, rows, k, X, ldx, ex, planes, kp);
    }
    oz2_count_launches(1);
    OZ2_CUDA_TRY(cudaGetLastError());
    return 0;
}
