// oz2_api.cu -- the C ABI of libozaki2 (include/ozaki2.h): argument checks, Step-1 constants,
// workspace carving and the launch sequence S1..S5 on the caller's stream.  No host synchronisation and no
// allocation on the ozaki2_dgemm path.
#include "../../include/ozaki2.h"
#include "oz2_common.cuh"

#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <atomic>
#include <mutex>
#include <string.h>
#include <vector>

static std::atomic<uint64_t> g_launches{0};
bool oz2_pdl_enabled()
{
    static const bool on = [] { const char *e = getenv("OZAKI2_PDL"); return !(e && e[0] == '0'); }();
    return on;
}
void oz2_count_launches(int n) { g_launches.fetch_add((uint64_t)n, std::memory_order_relaxed); }

namespace {

const int kModuli[OZ2_MAX_MODULI] = OZ2_MODULI_LIST;

// ---------------------------------------------------------------------------------------------
// small non-negative big integers, little-endian 32-bit limbs (host only, Step 1)
// ---------------------------------------------------------------------------------------------
typedef std::vector<uint32_t> Big;

Big big_from(uint32_t v) { return Big(1, v); }

void big_mul_small(Big &a, uint32_t f)
{
    uint64_t carry = 0;
    for (size_t t = 0; t < a.size(); t++) {
        uint64_t s = (uint64_t)a[t] * f + carry;
        a[t] = (uint32_t)s;
        carry = s >> 32;
    }
    if (carry) a.push_back((uint32_t)carry);
}

uint32_t big_mod_small(const Big &a, uint32_t p)
{
    uint64_t r = 0;
    for (size_t t = a.size(); t-- > 0;) r = ((r << 32) | a[t]) % p;
    return (uint32_t)r;
}

Big big_half(const Big &a)
{
    Big r(a.size());
    for (size_t t = 0; t < a.size(); t++) r[t] = (a[t] >> 1) | (t + 1 < a.size() ? a[t + 1] << 31 : 0u);
    return r;
}

long double big_to_ld(const Big &a)
{
    long double r = 0.0L;
    for (size_t t = a.size(); t-- > 0;) r = r * 4294967296.0L + (long double)a[t];
    return r;
}

void big_store(const Big &a, uint32_t *dst, int words)
{
    for (int t = 0; t < words; t++) dst[t] = t < (int)a.size() ? a[t] : 0u;
}

float f32_round_down(long double x)
{
    float f = (float)x;
    if ((long double)f > x) f = nextafterf(f, -INFINITY);
    return f;
}
float f32_round_up(long double x)
{
    float f = (float)x;
    if ((long double)f < x) f = nextafterf(f, INFINITY);
    return f;
}

int words_of_P_host(int N) { return N <= 4 ? 1 : N <= 8 ? 2 : N <= 12 ? 3 : N <= 16 ? 4 : 5; }

struct HostConsts {
    Oz2HostTables tab;
    int q[OZ2_MAX_MODULI + 1][OZ2_MAX_MODULI];
    Big P[OZ2_MAX_MODULI + 1];
    Big w[OZ2_MAX_MODULI + 1][OZ2_MAX_MODULI];
};

void build_host_consts(HostConsts &H)
{
    memset(&H.tab, 0, sizeof(H.tab));
    // ---- per-modulus tables
    for (int l = 0; l < OZ2_MAX_MODULI; l++) {
        Oz2ModTab &t = H.tab.mod[l];
        const uint32_t p = (uint32_t)kModuli[l];
        t.p = p;
        t.magic = (uint32_t)(0x100000000ull / p) + 1u;
        t.half = (p - 1) / 2;
        uint32_t pw = 1 % p;                               // 256^i mod p
        for (int i = 0; i < 12; i++) {
            t.wb[i / 4] |= pw << (8 * (i % 4));
            pw = (pw * 256u) % p;
        }
        t.conv_bias = 0;
        t.w16 = 65536u % p;
        t.epi_bias = ((32768u * t.w16 + p - 1) / p) * p;   // multiple of p, >= 2^15 w16
    }
    // ---- per-N tables
    for (int N = OZAKI2_MIN_MODULI; N <= OZ2_MAX_MODULI; N++) {
        Oz2CrtTab &c = H.tab.crt[N];
        Big P = big_from(1);
        for (int l = 0; l < N; l++) big_mul_small(P, (uint32_t)kModuli[l]);
        H.P[N] = P;
        const int nw = words_of_P_host(N);
        c.nw = nw;
        big_store(P, c.P, OZ2_MAX_WORDS);
        big_store(big_half(P), c.Phalf, OZ2_MAX_WORDS);
        for (int l = 0; l < N; l++) {
            Big Pl = big_from(1);
            for (int j = 0; j < N; j++)
                if (j != l) big_mul_small(Pl, (uint32_t)kModuli[j]);
            const uint32_t p = (uint32_t)kModuli[l];
            const uint32_t r = big_mod_small(Pl, p);
            uint32_t q = 0;
            for (uint32_t x = 1; x < p; x++)
                if ((r * x) % p == 1u) { q = x; break; }
            H.q[N][l] = (int)q;
            big_mul_small(Pl, q);                           // w_l = P_l q_l
            H.w[N][l] = Pl;
            big_store(Pl, c.w[l], OZ2_MAX_WORDS);
        }
        const long double Pld = big_to_ld(P);
        c.invP = (double)(ldexpl(1.0L, 32 * (nw - 1)) / Pld);
        Big Pm1 = P;
        Pm1[0] -= 1;                                        // P is a multiple of 256: no borrow
        const long double l2 = log2l(big_to_ld(Pm1));
        c.Pprop = f32_round_down(l2 / 2.0L - 0.5L);         // P:326-328 (= P'_accu)
        c.Pfast = f32_round_down(l2 / 2.0L - 1.5L);
        c.delta = f32_round_up(0.5L / (1.0L - ldexpl(1.0L, -22)));   // eq. (6)
    }
}

HostConsts &host_consts()
{
    static HostConsts H;
    static std::once_flag once;
    std::call_once(once, [] { build_host_consts(H); });
    return H;
}

// ---------------------------------------------------------------------------------------------
// per-device state
// ---------------------------------------------------------------------------------------------
constexpr int kMaxDevices = 64;
constexpr int kMaxPanels = 16;
struct DeviceState {
    bool tables_ready = false;
    bool checked = false;
    bool is_sm100 = false;
    void *ws = nullptr;
    size_t ws_bytes = 0;
    // ozaki2_dgemm_host: copy streams and ordering events (created on first use)
    bool host_ready = false;
    cudaStream_t s_h2d = nullptr, s_d2h = nullptr;
    cudaEvent_t ev0 = nullptr, evA = nullptr, evEnd = nullptr, evB[kMaxPanels] = {}, evC[kMaxPanels] = {};
};
DeviceState g_dev[kMaxDevices];
std::mutex g_mu;

int ensure_device(DeviceState **out)
{
    int dev = 0;
    OZ2_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return OZAKI2_ERR_DEVICE;
    std::lock_guard<std::mutex> lk(g_mu);
    DeviceState &d = g_dev[dev];
    if (!d.checked) {
        int major = 0;
        OZ2_CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
        d.is_sm100 = (major == 10);
        d.checked = true;
    }
    if (!d.is_sm100) return OZAKI2_ERR_DEVICE;
    if (!d.tables_ready) {
        const Oz2HostTables &t = host_consts().tab;
        int rc;
        if ((rc = oz2_scale_upload_tables(t))) return rc;
        if ((rc = oz2_convert_upload_tables(t))) return rc;
        if ((rc = oz2_gemm_upload_tables(t))) return rc;
        if ((rc = oz2_crt_upload_tables(t))) return rc;
        d.tables_ready = true;
    }
    *out = &d;
    return 0;
}

// ---------------------------------------------------------------------------------------------
// workspace layout
// ---------------------------------------------------------------------------------------------
struct Layout {
    int64_t kp, mp;
    size_t off_e, off_f, off_amax, off_ssq, off_EA, off_EB, off_rowmax, off_colmax, off_RA, off_RB, off_U, off_Abar,
        off_Bbar, total;
};

size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

Layout make_layout(int64_t m, int64_t n, int64_t k, int N, int mode)
{
    Layout L;
    L.kp = oz2_round_up(k > 0 ? k : 1, 128);
    L.mp = oz2_round_up(m > 0 ? m : 1, 16);
    size_t o = 0;
    L.off_e = o;      o = align_up(o + 4 * (size_t)m);
    L.off_f = o;      o = align_up(o + 4 * (size_t)n);
    L.off_amax = o;   o = align_up(o + 8 * (size_t)(m > n ? m : n));      // strided side: rows of A, or of B^T
    L.off_ssq = o;    o = align_up(o + 8 * (size_t)(m > n ? m : n));
    L.off_EA = o;     o = align_up(o + 4 * (size_t)m);
    L.off_EB = o;     o = align_up(o + 4 * (size_t)n);
    L.off_rowmax = o; o = align_up(o + 4 * (size_t)m);
    L.off_colmax = o; o = align_up(o + 4 * (size_t)n);
    L.off_RA = o;     o = align_up(o + (size_t)N * m * L.kp);
    L.off_RB = o;     o = align_up(o + (size_t)N * n * L.kp);
    L.off_U = o;      o = align_up(o + (size_t)N * n * L.mp);
    L.off_Abar = o;
    L.off_Bbar = o;
    if (mode == OZAKI2_MODE_ACCURATE) {
        o = align_up(o + (size_t)m * L.kp);
        L.off_Bbar = o;
        o = align_up(o + (size_t)n * L.kp);
    }
    L.total = o;
    return L;
}

// GEMM variant of the path: CTA pairs on 256 x 256 tiles (cta_group::2; measured 4 - 5 % faster than one CTA per
// 128 x 256 tile at 8192^3 under the board's power cap: a third less shared-memory fill per MMA), falling back to the
// single-CTA kernel for m <= 128 and K-blocked products.  OZAKI2_GEMM=single in the environment when the library is
// first used forces the single-CTA kernel (a tuning knob; results are identical).
int path_gemm_variant()
{
    static const int v = [] {
        const char *e = getenv("OZAKI2_GEMM");
        return (e && strcmp(e, "single") == 0) ? OZ2_GEMM_PATH : OZ2_GEMM_PAIR;
    }();
    return v;
}

// widths: fast / prop  <= floor(P'_prop) + 1 bits, accurate <= floor(P'_accu) + 7 bits; the narrow conversion format
// holds a' as a signed 64-bit integer, |a'| < 2^63
bool needs_wide_words(int N, int mode)
{
    const float Pp = host_consts().tab.crt[N].Pprop;
    const int width = (int)floorf(Pp) + (mode == OZAKI2_MODE_ACCURATE ? 7 : 1);
    return width > 63;
}

int check_args(int64_t m, int64_t n, int64_t k, const void *A, int64_t lda, const void *B, int64_t ldb,
               const void *C, int64_t ldc, int N, int mode, int transa = 0, int transb = 0)
{
    const int64_t rows_a = transa ? k : m, rows_b = transb ? n : k;
    if (m < 0) return -1;
    if (n < 0) return -2;
    if (k < 0 || k > OZAKI2_MAX_K) return -3;
    if (mode == OZAKI2_MODE_ACCURATE && k > OZAKI2_MAX_K_ACCURATE) return -3;
    if (m > 0 && k > 0 && !A) return -5;
    if (lda < (rows_a > 1 ? rows_a : 1)) return -6;
    if (n > 0 && k > 0 && !B) return -7;
    if (ldb < (rows_b > 1 ? rows_b : 1)) return -8;
    if (m > 0 && n > 0 && !C) return -10;
    if (ldc < (m > 1 ? m : 1)) return -11;
    if (N < OZAKI2_MIN_MODULI || N > OZAKI2_MAX_MODULI) return -12;
    if (mode != OZAKI2_MODE_ACCURATE && mode != OZAKI2_MODE_FAST && mode != OZAKI2_MODE_PROP) return -13;
    if (m > 0x7FFFFFFFll - 1024 || n > 0x7FFFFFFFll - 1024) return m > n ? -1 : -2;
    return 0;
}

template <typename T>
__global__ void k_scale_c(int64_t m, int64_t n, T beta, T *C, int64_t ldc)
{
    // one-dimensional grid of (row blocks) x n blocks: neither extent is bounded by the 65535 of grid.y / grid.z
    const int64_t nrb = (m + blockDim.x - 1) / blockDim.x;
    const int64_t j = blockIdx.x / nrb, i = (blockIdx.x - j * nrb) * blockDim.x + threadIdx.x;
    if (i < m) {
        T *p = C + i + j * ldc;
        *p = beta == (T)0 ? (T)0 : beta * *p;
    }
}

// blocks of a one-dimensional grid over (ceil(rows / 256) row blocks) x cols; the product is below 2^31 for anything
// that fits the device's memory (rows x cols elements are stored)
unsigned flat_grid(int64_t rows, int64_t cols) { return (unsigned)(((rows + 255) / 256) * cols); }

// ---- complex variants (DESIGN.md 8b #4): real embedding and the complex alpha / beta tail -----------
// R = double (zgemm) or float (cgemm); R2 = the interleaved pair type
template <typename R> struct Pair;
template <> struct Pair<double> { typedef double2 type; };
template <> struct Pair<float> { typedef float2 type; };
__device__ __forceinline__ double mul_rn(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double add_rn(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double sub_rn(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ float mul_rn(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float add_rn(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float sub_rn(float a, float b) { return __fsub_rn(a, b); }

// Atilde (2m x 2k) = [[A_r, -A_i], [A_i, A_r]] from interleaved complex A (m x k, lda complex elements)
template <typename R>
__global__ void k_zembed_a(int64_t m, int64_t k, const typename Pair<R>::type *__restrict__ A, int64_t lda, R *__restrict__ At)
{
    const int64_t nrb = (m + blockDim.x - 1) / blockDim.x;               // flat_grid(m, k)
    const int64_t h = blockIdx.x / nrb, i = (blockIdx.x - h * nrb) * blockDim.x + threadIdx.x;
    if (i >= m) return;
    const typename Pair<R>::type v = A[i + h * lda];
    const int64_t ld = 2 * m;
    At[i + h * ld] = v.x;
    At[i + (k + h) * ld] = -v.y;
    At[m + i + h * ld] = v.y;
    At[m + i + (k + h) * ld] = v.x;
}
// Btilde (2k x n) = [B_r; B_i]
template <typename R>
__global__ void k_zembed_b(int64_t k, int64_t n, const typename Pair<R>::type *__restrict__ B, int64_t ldb, R *__restrict__ Bt)
{
    const int64_t nrb = (k + blockDim.x - 1) / blockDim.x;               // flat_grid(k, n)
    const int64_t j = blockIdx.x / nrb, h = (blockIdx.x - j * nrb) * blockDim.x + threadIdx.x;
    if (h >= k) return;
    const typename Pair<R>::type v = B[h + j * ldb];
    Bt[h + j * 2 * k] = v.x;
    Bt[k + h + j * 2 * k] = v.y;
}
// C := alpha (c_r + i c_i) + beta C with [c_r; c_i] = Ct (2m x n); every product and sum rounded on its own, in the order
// stated in include/ozaki2.h; alpha == 1, beta == 0 and beta == 1 are not multiplied; have_c == 0: c = 0
template <typename R>
__global__ void k_zcombine(int64_t m, int64_t n, R ar, R ai, const R *__restrict__ Ct, int have_c, R br, R bi,
                           typename Pair<R>::type *__restrict__ C, int64_t ldc)
{
    const int64_t nrb = (m + blockDim.x - 1) / blockDim.x;               // flat_grid(m, n)
    const int64_t j = blockIdx.x / nrb, i = (blockIdx.x - j * nrb) * blockDim.x + threadIdx.x;
    if (i >= m) return;
    R tr = 0, ti = 0;
    if (have_c) {
        const R cr = Ct[i + j * 2 * m], ci = Ct[m + i + j * 2 * m];
        if (ar == (R)1 && ai == (R)0) { tr = cr; ti = ci; }
        else {
            tr = sub_rn(mul_rn(ar, cr), mul_rn(ai, ci));
            ti = add_rn(mul_rn(ar, ci), mul_rn(ai, cr));
        }
    }
    typename Pair<R>::type *dst = C + i + j * ldc;
    if (br == (R)1 && bi == (R)0) {                                    // beta == 1 is not multiplied: C is added as it is
        const typename Pair<R>::type c0 = *dst;
        tr = add_rn(tr, c0.x);
        ti = add_rn(ti, c0.y);
    } else if (br != (R)0 || bi != (R)0) {
        const typename Pair<R>::type c0 = *dst;
        tr = add_rn(tr, sub_rn(mul_rn(br, c0.x), mul_rn(bi, c0.y)));
        ti = add_rn(ti, add_rn(mul_rn(br, c0.y), mul_rn(bi, c0.x)));
    }
    typename Pair<R>::type o;
    o.x = tr; o.y = ti;
    *dst = o;
}

} // namespace

// =============================================================================================
// the path
// =============================================================================================
// f32 = 0: ozaki2_dgemm (A, B, C FP64); f32 = 1: ozaki2_sgemm (A, B, C FP32; alpha, beta hold floats)
// transa / transb != 0: the stored matrix is op(X)^T (k x m for A, n x k for B, column-major).  The vectors whose
// statistics and residues are needed -- rows of op(A), columns of op(B) -- are then contiguous for A and strided for
// B, i.e. the two movers / reductions simply swap sides.
static int run_path(int f32, int64_t m, int64_t n, int64_t k, double alpha, const void *A, int64_t lda, const void *B,
                    int64_t ldb, double beta, void *C, int64_t ldc, int N, int mode, cudaStream_t st,
                    const ozaki2_stage_outputs *out, int transa = 0, int transb = 0, void *call_ws = nullptr, size_t call_ws_bytes = 0,
                    bool use_call_ws = false)
{
    int rc = check_args(m, n, k, A, lda, B, ldb, C, ldc, N, mode, transa, transb);
    const int strided_a = transa ? 0 : 1, strided_b = transb ? 1 : 0;
    if (rc) return rc;
    if (m == 0 || n == 0) return 0;
    DeviceState *dev = nullptr;
    if ((rc = ensure_device(&dev))) return rc;
    if (k == 0 || alpha == 0.0) {
        // C := beta C (zeros if beta == 0, BLAS rule)
        if (!(beta == 1.0)) {
            const dim3 grid(flat_grid(m, n));
            if (f32) k_scale_c<float><<<grid, 256, 0, st>>>(m, n, (float)beta, static_cast<float *>(C), ldc);
            else k_scale_c<double><<<grid, 256, 0, st>>>(m, n, beta, static_cast<double *>(C), ldc);
            oz2_count_launches(1);
            OZ2_CUDA_TRY(cudaGetLastError());
        }
        return 0;
    }
    const Layout L = make_layout(m, n, k, N, mode);
    // the workspace of this call: the caller's own (ozaki2_*gemm_ws) or the one registered for the device
    void *ws_ptr = use_call_ws ? call_ws : dev->ws;
    const size_t ws_have = use_call_ws ? call_ws_bytes : dev->ws_bytes;
    if (!ws_ptr || ws_have < L.total || (reinterpret_cast<uintptr_t>(ws_ptr) & 255)) return OZAKI2_ERR_WORKSPACE;
    uint8_t *ws = static_cast<uint8_t *>(ws_ptr);
    int32_t *e = reinterpret_cast<int32_t *>(ws + L.off_e), *f = reinterpret_cast<int32_t *>(ws + L.off_f);
    unsigned long long *amax = reinterpret_cast<unsigned long long *>(ws + L.off_amax);
    unsigned long long *ssq = reinterpret_cast<unsigned long long *>(ws + L.off_ssq);
    int32_t *EA = reinterpret_cast<int32_t *>(ws + L.off_EA), *EB = reinterpret_cast<int32_t *>(ws + L.off_EB);
    int32_t *rowmax = reinterpret_cast<int32_t *>(ws + L.off_rowmax), *colmax = reinterpret_cast<int32_t *>(ws + L.off_colmax);
    int8_t *RA = reinterpret_cast<int8_t *>(ws + L.off_RA), *RB = reinterpret_cast<int8_t *>(ws + L.off_RB);
    uint8_t *U = ws + L.off_U;

    struct StageEvents {                                    // destroyed on every exit path
        cudaEvent_t ev[5] = { nullptr, nullptr, nullptr, nullptr, nullptr };
        ~StageEvents() { for (int t = 0; t < 5; t++) if (ev[t]) cudaEventDestroy(ev[t]); }
    } sev;
    cudaEvent_t *ev = sev.ev;
    const bool timing = out && out->stage_ms;
    cudaEvent_t *uev = out && out->stage_events ? reinterpret_cast<cudaEvent_t *>(out->stage_events) : nullptr;
    if (timing) {
        for (int t = 0; t < 5; t++) OZ2_CUDA_TRY(cudaEventCreate(&ev[t]));
        OZ2_CUDA_TRY(cudaEventRecord(ev[0], st));
    }
    if (uev) OZ2_CUDA_TRY(cudaEventRecord(uev[0], st));
    // ---- S1 scaling
    if (mode == OZAKI2_MODE_ACCURATE) {
        int8_t *Abar = reinterpret_cast<int8_t *>(ws + L.off_Abar), *Bbar = reinterpret_cast<int8_t *>(ws + L.off_Bbar);
        OZ2_CUDA_TRY(cudaMemsetAsync(rowmax, 0, sizeof(int32_t) * (size_t)m, st));
        OZ2_CUDA_TRY(cudaMemsetAsync(colmax, 0, sizeof(int32_t) * (size_t)n, st));
        if ((rc = oz2_launch_scale_accu_side(f32, strided_a, m, k, A, lda, amax, EA, Abar, L.kp, st))) return rc;
        if ((rc = oz2_launch_scale_accu_side(f32, strided_b, n, k, B, ldb, amax, EB, Bbar, L.kp, st))) return rc;
        if ((rc = oz2_launch_gemm_tc(path_gemm_variant(), 1, 0, m, n, k, Abar, Bbar, L.kp, nullptr, L.mp, rowmax, colmax, st))) return rc;
        if ((rc = oz2_launch_scale_accu_finish(N, m, n, EA, EB, rowmax, colmax, e, f, st))) return rc;
    } else {
        if (strided_a) rc = oz2_launch_scale_rows(mode, N, f32, m, k, A, lda, amax, ssq, e, st);
        else rc = oz2_launch_scale_cols(mode, N, f32, m, k, A, lda, e, st);
        if (rc) return rc;
        if (strided_b) rc = oz2_launch_scale_rows(mode, N, f32, n, k, B, ldb, amax, ssq, f, st);
        else rc = oz2_launch_scale_cols(mode, N, f32, n, k, B, ldb, f, st);
        if (rc) return rc;
    }
    if (timing) OZ2_CUDA_TRY(cudaEventRecord(ev[1], st));
    if (uev) OZ2_CUDA_TRY(cudaEventRecord(uev[1], st));
    // ---- S2 conversion
    const int wide = needs_wide_words(N, mode) ? 1 : 0;
    if ((rc = oz2_launch_convert(strided_a ? 0 : 1, N, wide, f32, m, k, A, lda, e, RA, L.kp, st))) return rc;
    if ((rc = oz2_launch_convert(strided_b ? 0 : 1, N, wide, f32, n, k, B, ldb, f, RB, L.kp, st))) return rc;
    if (timing) OZ2_CUDA_TRY(cudaEventRecord(ev[2], st));
    if (uev) OZ2_CUDA_TRY(cudaEventRecord(uev[2], st));
    // ---- S3 residue GEMMs
    if ((rc = oz2_launch_gemm_tc(path_gemm_variant(), N, 0, m, n, k, RA, RB, L.kp, U, L.mp, nullptr, nullptr, st))) return rc;
    if (timing) OZ2_CUDA_TRY(cudaEventRecord(ev[3], st));
    if (uev) OZ2_CUDA_TRY(cudaEventRecord(uev[3], st));
    // ---- S4 + S5
    if ((rc = oz2_launch_crt(N, f32, m, n, U, L.mp, e, f, alpha, beta, C, ldc, out ? out->Cpp : nullptr, st))) return rc;
    if (timing) OZ2_CUDA_TRY(cudaEventRecord(ev[4], st));
    if (uev) OZ2_CUDA_TRY(cudaEventRecord(uev[4], st));

    if (out) {
        if (out->e) OZ2_CUDA_TRY(cudaMemcpyAsync(out->e, e, 4 * (size_t)m, cudaMemcpyDeviceToDevice, st));
        if (out->f) OZ2_CUDA_TRY(cudaMemcpyAsync(out->f, f, 4 * (size_t)n, cudaMemcpyDeviceToDevice, st));
        if (mode == OZAKI2_MODE_ACCURATE) {
            if (out->rowmax) OZ2_CUDA_TRY(cudaMemcpyAsync(out->rowmax, rowmax, 4 * (size_t)m, cudaMemcpyDeviceToDevice, st));
            if (out->colmax) OZ2_CUDA_TRY(cudaMemcpyAsync(out->colmax, colmax, 4 * (size_t)n, cudaMemcpyDeviceToDevice, st));
        }
        // pitched internal planes -> canonical dense layouts
        if (out->resA)
            OZ2_CUDA_TRY(cudaMemcpy2DAsync(out->resA, (size_t)k, RA, (size_t)L.kp, (size_t)k, (size_t)N * m, cudaMemcpyDeviceToDevice, st));
        if (out->resB)
            OZ2_CUDA_TRY(cudaMemcpy2DAsync(out->resB, (size_t)k, RB, (size_t)L.kp, (size_t)k, (size_t)N * n, cudaMemcpyDeviceToDevice, st));
        if (out->U)
            OZ2_CUDA_TRY(cudaMemcpy2DAsync(out->U, (size_t)m, U, (size_t)L.mp, (size_t)m, (size_t)N * n, cudaMemcpyDeviceToDevice, st));
        if (timing) {
            OZ2_CUDA_TRY(cudaStreamSynchronize(st));
            for (int t = 0; t < 4; t++) OZ2_CUDA_TRY(cudaEventElapsedTime(out->stage_ms + t, ev[t], ev[t + 1]));
            OZ2_CUDA_TRY(cudaEventElapsedTime(out->stage_ms + 4, ev[0], ev[4]));
        }
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// ozaki2_dgemm_host, modes 1 and 2: column panels of B / C so that the H2D copy of panel p+1 and the D2H copy of
// panel p-1 overlap the kernels of panel p.  (e_i depends on row i of A only and f_j on column j of B only, so a
// panel is the same computation as the monolithic call; accurate mode needs all of B before any e_i and takes the
// plain route.)  Kernels run on the caller's stream in order, so all panels share one workspace.
// ---------------------------------------------------------------------------------------------
static int ensure_host_streams(DeviceState *d)
{
    std::lock_guard<std::mutex> lk(g_mu);
    if (d->host_ready) return 0;
    OZ2_CUDA_TRY(cudaStreamCreateWithFlags(&d->s_h2d, cudaStreamNonBlocking));
    OZ2_CUDA_TRY(cudaStreamCreateWithFlags(&d->s_d2h, cudaStreamNonBlocking));
    OZ2_CUDA_TRY(cudaEventCreateWithFlags(&d->ev0, cudaEventDisableTiming));
    OZ2_CUDA_TRY(cudaEventCreateWithFlags(&d->evA, cudaEventDisableTiming));
    OZ2_CUDA_TRY(cudaEventCreateWithFlags(&d->evEnd, cudaEventDisableTiming));
    for (int p = 0; p < kMaxPanels; p++) {
        OZ2_CUDA_TRY(cudaEventCreateWithFlags(&d->evB[p], cudaEventDisableTiming));
        OZ2_CUDA_TRY(cudaEventCreateWithFlags(&d->evC[p], cudaEventDisableTiming));
    }
    d->host_ready = true;
    return 0;
}

// the enqueue part of the panel pipeline; esz = bytes per element (8: FP64, 4: FP32)
static int host_pipelined_enqueue(int f32, int64_t m, int64_t n, int64_t k, double alpha, const uint8_t *A_host, int64_t lda,
                                  const uint8_t *B_host, int64_t ldb, double beta, uint8_t *C_host, int64_t ldc, int N, int mode,
                                  uint8_t *dA, uint8_t *dB, uint8_t *dC, cudaStream_t st, DeviceState *dev)
{
    int rc;
    const size_t esz = f32 ? 4 : 8;
    const Layout L = make_layout(m, n, k, N, mode);
    if (!dev->ws || dev->ws_bytes < L.total) return OZAKI2_ERR_WORKSPACE;
    uint8_t *ws = static_cast<uint8_t *>(dev->ws);
    int32_t *e = reinterpret_cast<int32_t *>(ws + L.off_e), *f = reinterpret_cast<int32_t *>(ws + L.off_f);
    unsigned long long *amax = reinterpret_cast<unsigned long long *>(ws + L.off_amax);
    unsigned long long *ssq = reinterpret_cast<unsigned long long *>(ws + L.off_ssq);
    int8_t *RA = reinterpret_cast<int8_t *>(ws + L.off_RA), *RB = reinterpret_cast<int8_t *>(ws + L.off_RB);
    uint8_t *U = ws + L.off_U;
    const int wide = needs_wide_words(N, mode) ? 1 : 0;
    // panels: multiples of 256 columns (the GEMM tile), at most kMaxPanels.  What cannot overlap the copies is the last panel's
    // kernels and its copy back, so the panels are small: at 8192^3, 4 / 8 / 16 / 32 panels measured 24.4 / 23.0 / 22.3 / 22.6+ ms
    int64_t np = oz2_round_up((n + kMaxPanels - 1) / kMaxPanels, 256);
    const int panels = (int)((n + np - 1) / np);
    cudaStream_t sh = dev->s_h2d, sd = dev->s_d2h;
    OZ2_CUDA_TRY(cudaEventRecord(dev->ev0, st));
    OZ2_CUDA_TRY(cudaStreamWaitEvent(sh, dev->ev0, 0));
    OZ2_CUDA_TRY(cudaStreamWaitEvent(sd, dev->ev0, 0));
    // ---- copies in: A, then the panels of B (and of C if it is read)
    OZ2_CUDA_TRY(cudaMemcpy2DAsync(dA, esz * (size_t)m, A_host, esz * (size_t)lda, esz * (size_t)m, (size_t)k, cudaMemcpyHostToDevice, sh));
    OZ2_CUDA_TRY(cudaEventRecord(dev->evA, sh));
    for (int p = 0; p < panels; p++) {
        const int64_t j0 = p * np, nc = (j0 + np < n ? np : n - j0);
        OZ2_CUDA_TRY(cudaMemcpy2DAsync(dB + esz * (size_t)(j0 * k), esz * (size_t)k, B_host + esz * (size_t)(j0 * ldb), esz * (size_t)ldb,
                                       esz * (size_t)k, (size_t)nc, cudaMemcpyHostToDevice, sh));
        if (beta != 0.0)
            OZ2_CUDA_TRY(cudaMemcpy2DAsync(dC + esz * (size_t)(j0 * m), esz * (size_t)m, C_host + esz * (size_t)(j0 * ldc), esz * (size_t)ldc,
                                           esz * (size_t)m, (size_t)nc, cudaMemcpyHostToDevice, sh));
        OZ2_CUDA_TRY(cudaEventRecord(dev->evB[p], sh));
    }
    // ---- rows of A: S1, S2
    OZ2_CUDA_TRY(cudaStreamWaitEvent(st, dev->evA, 0));
    if ((rc = oz2_launch_scale_rows(mode, N, f32, m, k, dA, m, amax, ssq, e, st))) return rc;
    if ((rc = oz2_launch_convert(0, N, wide, f32, m, k, dA, m, e, RA, L.kp, st))) return rc;
    // ---- panels: S1, S2 of the columns, S3, S4 + S5, copy out
    for (int p = 0; p < panels; p++) {
        const int64_t j0 = p * np, nc = (j0 + np < n ? np : n - j0);
        OZ2_CUDA_TRY(cudaStreamWaitEvent(st, dev->evB[p], 0));
        if ((rc = oz2_launch_scale_cols(mode, N, f32, nc, k, dB + esz * (size_t)(j0 * k), k, f, st))) return rc;
        if ((rc = oz2_launch_convert(1, N, wide, f32, nc, k, dB + esz * (size_t)(j0 * k), k, f, RB, L.kp, st))) return rc;
        if ((rc = oz2_launch_gemm_tc(path_gemm_variant(), N, 0, m, nc, k, RA, RB, L.kp, U, L.mp, nullptr, nullptr, st))) return rc;
        if ((rc = oz2_launch_crt(N, f32, m, nc, U, L.mp, e, f, alpha, beta, dC + esz * (size_t)(j0 * m), m, nullptr, st))) return rc;
        OZ2_CUDA_TRY(cudaEventRecord(dev->evC[p], st));
        OZ2_CUDA_TRY(cudaStreamWaitEvent(sd, dev->evC[p], 0));
        OZ2_CUDA_TRY(cudaMemcpy2DAsync(C_host + esz * (size_t)(j0 * ldc), esz * (size_t)ldc, dC + esz * (size_t)(j0 * m), esz * (size_t)m,
                                       esz * (size_t)m, (size_t)nc, cudaMemcpyDeviceToHost, sd));
    }
    OZ2_CUDA_TRY(cudaEventRecord(dev->evEnd, sd));
    OZ2_CUDA_TRY(cudaStreamWaitEvent(st, dev->evEnd, 0));
    return 0;
}

static int host_pipelined(int f32, int64_t m, int64_t n, int64_t k, double alpha, const uint8_t *A_host, int64_t lda,
                          const uint8_t *B_host, int64_t ldb, double beta, uint8_t *C_host, int64_t ldc, int N, int mode,
                          uint8_t *dA, uint8_t *dB, uint8_t *dC, cudaStream_t st, DeviceState *dev)
{
    int rc;
    if ((rc = ensure_host_streams(dev))) return rc;
    rc = host_pipelined_enqueue(f32, m, n, k, alpha, A_host, lda, B_host, ldb, beta, C_host, ldc, N, mode, dA, dB, dC, st, dev);
    // success or not, nothing may still be reading or writing the caller's host buffers when this returns
    const cudaError_t e1 = cudaStreamSynchronize(dev->s_h2d), e2 = cudaStreamSynchronize(dev->s_d2h), e3 = cudaStreamSynchronize(st);
    if (rc) return rc;
    if (e1 != cudaSuccess) return (int)e1;
    if (e2 != cudaSuccess) return (int)e2;
    return (int)e3;
}

// ozaki2_dgemm_host / ozaki2_sgemm_host
static int host_entry(int f32, int64_t m, int64_t n, int64_t k, double alpha, const void *A_host, int64_t lda, const void *B_host,
                      int64_t ldb, double beta, void *C_host, int64_t ldc, int num_moduli, int scaling_mode, void *device_scratch,
                      size_t scratch_bytes, cudaStream_t st)
{
    int rc = check_args(m, n, k, A_host, lda, B_host, ldb, C_host, ldc, num_moduli, scaling_mode);
    if (rc) return rc;
    if (m == 0 || n == 0) return 0;
    const size_t esz = f32 ? 4 : 8;
    const size_t need = align_up(esz * (size_t)m * k) + align_up(esz * (size_t)k * n) + align_up(esz * (size_t)m * n);
    if (!device_scratch || scratch_bytes < need) return -14;
    uint8_t *base = static_cast<uint8_t *>(device_scratch);
    uint8_t *dA = base, *dB = base + align_up(esz * (size_t)m * k), *dC = dB + align_up(esz * (size_t)k * n);
    const uint8_t *Ah = static_cast<const uint8_t *>(A_host), *Bh = static_cast<const uint8_t *>(B_host);
    uint8_t *Ch = static_cast<uint8_t *>(C_host);
    if (k > 0 && alpha != 0.0 && scaling_mode != OZAKI2_MODE_ACCURATE && n >= 512) {
        DeviceState *dev = nullptr;
        if ((rc = ensure_device(&dev))) return rc;
        return host_pipelined(f32, m, n, k, alpha, Ah, lda, Bh, ldb, beta, Ch, ldc, num_moduli, scaling_mode, dA, dB, dC, st, dev);
    }
    auto enqueue = [&]() -> int {
        if (k > 0) {
            OZ2_CUDA_TRY(cudaMemcpy2DAsync(dA, esz * (size_t)m, Ah, esz * (size_t)lda, esz * (size_t)m, (size_t)k, cudaMemcpyHostToDevice, st));
            OZ2_CUDA_TRY(cudaMemcpy2DAsync(dB, esz * (size_t)k, Bh, esz * (size_t)ldb, esz * (size_t)k, (size_t)n, cudaMemcpyHostToDevice, st));
        }
        if (beta != 0.0)
            OZ2_CUDA_TRY(cudaMemcpy2DAsync(dC, esz * (size_t)m, Ch, esz * (size_t)ldc, esz * (size_t)m, (size_t)n, cudaMemcpyHostToDevice, st));
        const int r = run_path(f32, m, n, k, alpha, dA, m > 1 ? m : 1, dB, k > 1 ? k : 1, beta, dC, m > 1 ? m : 1, num_moduli, scaling_mode, st, nullptr);
        if (r) return r;
        OZ2_CUDA_TRY(cudaMemcpy2DAsync(Ch, esz * (size_t)ldc, dC, esz * (size_t)m, esz * (size_t)m, (size_t)n, cudaMemcpyDeviceToHost, st));
        return 0;
    };
    rc = enqueue();
    const cudaError_t es = cudaStreamSynchronize(st);      // also on error: the host buffers must be quiescent on return
    if (rc) return rc;
    return (int)es;
}

// BLAS-style flags: 'N' / 'T' / 'C' (any case; 'C' = 'T' for real matrices) or the CBLAS enums 111 / 112 / 113
static int parse_trans(int c)
{
    if (c == 'N' || c == 'n' || c == 111) return 0;
    if (c == 'T' || c == 't' || c == 'C' || c == 'c' || c == 112 || c == 113) return 1;
    return -1;
}
// 'C' column-major / 'R' row-major (any case) or the CBLAS enums 102 / 101
static int parse_layout(int c)
{
    if (c == 'C' || c == 'c' || c == 102) return 0;
    if (c == 'R' || c == 'r' || c == 101) return 1;
    return -1;
}

// The full BLAS shape.  A row-major problem is the column-major problem C^T = op(B)^T op(A)^T on the same memory:
// the operands swap places and m, n swap, the flags stay with their matrices.  The vectors the method scales --
// rows of op(A), columns of op(B) -- are the same vectors in both views, so the result is the oracle's on the
// logical matrices bit for bit.
static int blas_entry(int f32, int layout, int transa, int transb, int64_t m, int64_t n, int64_t k, double alpha, const void *A,
                      int64_t lda, const void *B, int64_t ldb, double beta, void *C, int64_t ldc, int N, int mode, cudaStream_t st)
{
    const int lay = parse_layout(layout), ta = parse_trans(transa), tb = parse_trans(transb);
    if (lay < 0) return -1;
    if (ta < 0) return -2;
    if (tb < 0) return -3;
    int rc;
    if (!lay) rc = run_path(f32, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc, N, mode, st, nullptr, ta, tb);
    else rc = run_path(f32, n, m, k, alpha, B, ldb, A, lda, beta, C, ldc, N, mode, st, nullptr, tb, ta);
    if (rc >= 0 || rc <= -100) return rc;
    // argument numbers of run_path (m n k alpha A lda B ldb beta C ldc N mode stream) -> this prototype
    static const int col[15] = { 0, 4, 5, 6, 7, 8, 9, 10, 11, 12, 13, 14, 15, 16, 17 };
    static const int row[15] = { 0, 5, 4, 6, 7, 10, 11, 8, 9, 12, 13, 14, 15, 16, 17 };
    return -(lay ? row[-rc] : col[-rc]);
}

static size_t complex_workspace_bytes(size_t esz, int64_t m, int64_t n, int64_t k, int num_moduli, int scaling_mode)
{
    if (m < 0 || n < 0 || k < 0 || 2 * k > OZAKI2_MAX_K) return 0;
    const size_t real_ws = ozaki2_workspace_bytes(2 * m, n, 2 * k, num_moduli, scaling_mode);
    if (!real_ws && m && n && k) return 0;
    return align_up(real_ws) + align_up(esz * (size_t)(2 * m) * (2 * k)) + align_up(esz * (size_t)(2 * k) * n) + align_up(esz * (size_t)(2 * m) * n);
}

// ozaki2_zgemm (R = double) / ozaki2_cgemm (R = float): embed, run the real path, combine
template <typename R>
static int complex_entry(int64_t m, int64_t n, int64_t k, R alpha_re, R alpha_im, const R *A, int64_t lda, const R *B, int64_t ldb,
                         R beta_re, R beta_im, R *C, int64_t ldc, int num_moduli, int scaling_mode, void *stream)
{
    typedef typename Pair<R>::type R2;
    constexpr size_t esz = sizeof(R);
    constexpr uintptr_t amask = 2 * sizeof(R) - 1;                     // interleaved pairs: 16-byte (FP64) / 8-byte (FP32) aligned
    if (m < 0) return -1;
    if (n < 0) return -2;
    if (k < 0 || 2 * k > OZAKI2_MAX_K || (scaling_mode == OZAKI2_MODE_ACCURATE && 2 * k > OZAKI2_MAX_K_ACCURATE)) return -3;
    if (m > 0 && k > 0 && (!A || (reinterpret_cast<uintptr_t>(A) & amask))) return -6;
    if (lda < (m > 1 ? m : 1)) return -7;
    if (n > 0 && k > 0 && (!B || (reinterpret_cast<uintptr_t>(B) & amask))) return -8;
    if (ldb < (k > 1 ? k : 1)) return -9;
    if (m > 0 && n > 0 && (!C || (reinterpret_cast<uintptr_t>(C) & amask))) return -12;
    if (ldc < (m > 1 ? m : 1)) return -13;
    if (num_moduli < OZAKI2_MIN_MODULI || num_moduli > OZAKI2_MAX_MODULI) return -14;
    if (scaling_mode < 0 || scaling_mode > 2) return -15;
    if (m > (0x7FFFFFFFll - 1024) / 2 || n > 0x7FFFFFFFll - 1024) return m > n ? -1 : -2;
    if (m == 0 || n == 0) return 0;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    DeviceState *dev = nullptr;
    int rc = ensure_device(&dev);
    if (rc) return rc;
    const dim3 gc(flat_grid(m, n));
    const bool have_c = k > 0 && !(alpha_re == (R)0 && alpha_im == (R)0);
    if (!have_c) {
        if (beta_re == (R)1 && beta_im == (R)0) return 0;               // C := C, the BLAS quick return: C is not touched
        k_zcombine<R><<<gc, 256, 0, st>>>(m, n, alpha_re, alpha_im, nullptr, 0, beta_re, beta_im, reinterpret_cast<R2 *>(C), ldc);
        oz2_count_launches(1);
        OZ2_CUDA_TRY(cudaGetLastError());
        return 0;
    }
    const size_t real_ws = align_up(make_layout(2 * m, n, 2 * k, num_moduli, scaling_mode).total);
    if (!dev->ws || dev->ws_bytes < complex_workspace_bytes(esz, m, n, k, num_moduli, scaling_mode)) return OZAKI2_ERR_WORKSPACE;
    uint8_t *ws = static_cast<uint8_t *>(dev->ws);
    R *At = reinterpret_cast<R *>(ws + real_ws);
    R *Bt = reinterpret_cast<R *>(ws + real_ws + align_up(esz * (size_t)(2 * m) * (2 * k)));
    R *Ct = reinterpret_cast<R *>(ws + real_ws + align_up(esz * (size_t)(2 * m) * (2 * k)) + align_up(esz * (size_t)(2 * k) * n));
    k_zembed_a<R><<<dim3(flat_grid(m, k)), 256, 0, st>>>(m, k, reinterpret_cast<const R2 *>(A), lda, At);
    OZ2_CUDA_TRY(cudaGetLastError());
    k_zembed_b<R><<<dim3(flat_grid(k, n)), 256, 0, st>>>(k, n, reinterpret_cast<const R2 *>(B), ldb, Bt);
    OZ2_CUDA_TRY(cudaGetLastError());
    oz2_count_launches(2);
    rc = run_path(esz == 4 ? 1 : 0, 2 * m, n, 2 * k, 1.0, At, 2 * m, Bt, 2 * k, 0.0, Ct, 2 * m, num_moduli, scaling_mode, st, nullptr);
    if (rc) return rc < 0 && rc > -100 ? -100 - rc : rc;      // an argument error of the embedded call would be a bug here
    k_zcombine<R><<<gc, 256, 0, st>>>(m, n, alpha_re, alpha_im, Ct, 1, beta_re, beta_im, reinterpret_cast<R2 *>(C), ldc);
    oz2_count_launches(1);
    OZ2_CUDA_TRY(cudaGetLastError());
    return 0;
}

extern "C" {

int ozaki2_dgemm(int64_t m, int64_t n, int64_t k, double alpha, const double *A, int64_t lda, const double *B,
                 int64_t ldb, double beta, double *C, int64_t ldc, int num_moduli, int scaling_mode, void *stream)
{
    return run_path(0, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc, num_moduli, scaling_mode,
                    static_cast<cudaStream_t>(stream), nullptr);
}

int ozaki2_dgemm_ws(int64_t m, int64_t n, int64_t k, double alpha, const double *A, int64_t lda, const double *B,
                    int64_t ldb, double beta, double *C, int64_t ldc, int num_moduli, int scaling_mode, void *workspace,
                    size_t workspace_bytes, void *stream)
{
    const int rc = run_path(0, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc, num_moduli, scaling_mode,
                            static_cast<cudaStream_t>(stream), nullptr, 0, 0, workspace, workspace_bytes, true);
    return rc == OZAKI2_ERR_WORKSPACE ? -14 : rc;          // here the workspace is the 14th argument
}

int ozaki2_sgemm_ws(int64_t m, int64_t n, int64_t k, float alpha, const float *A, int64_t lda, const float *B,
                    int64_t ldb, float beta, float *C, int64_t ldc, int num_moduli, int scaling_mode, void *workspace,
                    size_t workspace_bytes, void *stream)
{
    const int rc = run_path(1, m, n, k, (double)alpha, A, lda, B, ldb, (double)beta, C, ldc, num_moduli, scaling_mode,
                            static_cast<cudaStream_t>(stream), nullptr, 0, 0, workspace, workspace_bytes, true);
    return rc == OZAKI2_ERR_WORKSPACE ? -14 : rc;
}

int ozaki2_dgemm_stages(int64_t m, int64_t n, int64_t k, double alpha, const double *A, int64_t lda, const double *B,
                        int64_t ldb, double beta, double *C, int64_t ldc, int num_moduli, int scaling_mode, void *stream,
                        const ozaki2_stage_outputs *out)
{
    return run_path(0, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc, num_moduli, scaling_mode,
                    static_cast<cudaStream_t>(stream), out);
}

int ozaki2_sgemm(int64_t m, int64_t n, int64_t k, float alpha, const float *A, int64_t lda, const float *B, int64_t ldb,
                 float beta, float *C, int64_t ldc, int num_moduli, int scaling_mode, void *stream)
{
    return run_path(1, m, n, k, (double)alpha, A, lda, B, ldb, (double)beta, C, ldc, num_moduli, scaling_mode,
                    static_cast<cudaStream_t>(stream), nullptr);
}

int ozaki2_sgemm_stages(int64_t m, int64_t n, int64_t k, float alpha, const float *A, int64_t lda, const float *B,
                        int64_t ldb, float beta, float *C, int64_t ldc, int num_moduli, int scaling_mode, void *stream,
                        const ozaki2_stage_outputs *out)
{
    return run_path(1, m, n, k, (double)alpha, A, lda, B, ldb, (double)beta, C, ldc, num_moduli, scaling_mode,
                    static_cast<cudaStream_t>(stream), out);
}

int ozaki2_dgemm_t(int transa, int transb, int64_t m, int64_t n, int64_t k, double alpha, const double *A, int64_t lda,
                   const double *B, int64_t ldb, double beta, double *C, int64_t ldc, int num_moduli, int scaling_mode,
                   void *stream)
{
    if (transa != 0 && transa != 1) return -1;
    if (transb != 0 && transb != 1) return -2;
    const int rc = run_path(0, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc, num_moduli, scaling_mode,
                            static_cast<cudaStream_t>(stream), nullptr, transa, transb);
    return rc < 0 && rc > -100 ? rc - 2 : rc;              // argument numbers shift by the two leading flags
}

size_t ozaki2_workspace_bytes(int64_t m, int64_t n, int64_t k, int num_moduli, int scaling_mode)
{
    if (m < 0 || n < 0 || k < 0 || k > OZAKI2_MAX_K) return 0;
    if (num_moduli < OZAKI2_MIN_MODULI || num_moduli > OZAKI2_MAX_MODULI) return 0;
    if (scaling_mode < 0 || scaling_mode > 2) return 0;
    return make_layout(m, n, k, num_moduli, scaling_mode).total;
}

// a row-major ozaki2_*gemm_blas call runs as the (n, m, k) problem, and the layout is not symmetric in m and n
// (U is N n round_up(m, 16) bytes)
size_t ozaki2_blas_workspace_bytes(int layout, int64_t m, int64_t n, int64_t k, int num_moduli, int scaling_mode)
{
    const int lay = parse_layout(layout);
    if (lay < 0) return 0;
    return lay ? ozaki2_workspace_bytes(n, m, k, num_moduli, scaling_mode) : ozaki2_workspace_bytes(m, n, k, num_moduli, scaling_mode);
}

int ozaki2_set_workspace(void *device_ptr, size_t bytes)
{
    int dev = 0;
    OZ2_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return OZAKI2_ERR_DEVICE;
    if (device_ptr && (reinterpret_cast<uintptr_t>(device_ptr) & 255)) return -1;
    if (!device_ptr && bytes) return -2;
    std::lock_guard<std::mutex> lk(g_mu);
    g_dev[dev].ws = device_ptr;
    g_dev[dev].ws_bytes = device_ptr ? bytes : 0;
    return 0;
}

size_t ozaki2_host_scratch_bytes(int64_t m, int64_t n, int64_t k)
{
    if (m < 0 || n < 0 || k < 0) return 0;
    return align_up(8 * (size_t)m * k) + align_up(8 * (size_t)k * n) + align_up(8 * (size_t)m * n);
}

int ozaki2_dgemm_host(int64_t m, int64_t n, int64_t k, double alpha, const double *A_host, int64_t lda,
                      const double *B_host, int64_t ldb, double beta, double *C_host, int64_t ldc, int num_moduli,
                      int scaling_mode, void *device_scratch, size_t scratch_bytes, void *stream)
{
    return host_entry(0, m, n, k, alpha, A_host, lda, B_host, ldb, beta, C_host, ldc, num_moduli, scaling_mode, device_scratch,
                      scratch_bytes, static_cast<cudaStream_t>(stream));
}

int ozaki2_sgemm_host(int64_t m, int64_t n, int64_t k, float alpha, const float *A_host, int64_t lda, const float *B_host,
                      int64_t ldb, float beta, float *C_host, int64_t ldc, int num_moduli, int scaling_mode,
                      void *device_scratch, size_t scratch_bytes, void *stream)
{
    return host_entry(1, m, n, k, (double)alpha, A_host, lda, B_host, ldb, (double)beta, C_host, ldc, num_moduli, scaling_mode,
                      device_scratch, scratch_bytes, static_cast<cudaStream_t>(stream));
}

int ozaki2_sgemm_t(int transa, int transb, int64_t m, int64_t n, int64_t k, float alpha, const float *A, int64_t lda,
                   const float *B, int64_t ldb, float beta, float *C, int64_t ldc, int num_moduli, int scaling_mode, void *stream)
{
    if (transa != 0 && transa != 1) return -1;
    if (transb != 0 && transb != 1) return -2;
    const int rc = run_path(1, m, n, k, (double)alpha, A, lda, B, ldb, (double)beta, C, ldc, num_moduli, scaling_mode,
                            static_cast<cudaStream_t>(stream), nullptr, transa, transb);
    return rc < 0 && rc > -100 ? rc - 2 : rc;
}

int ozaki2_dgemm_blas(int layout, int transa, int transb, int64_t m, int64_t n, int64_t k, double alpha, const double *A,
                      int64_t lda, const double *B, int64_t ldb, double beta, double *C, int64_t ldc, int num_moduli,
                      int scaling_mode, void *stream)
{
    return blas_entry(0, layout, transa, transb, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc, num_moduli, scaling_mode,
                      static_cast<cudaStream_t>(stream));
}

int ozaki2_sgemm_blas(int layout, int transa, int transb, int64_t m, int64_t n, int64_t k, float alpha, const float *A,
                      int64_t lda, const float *B, int64_t ldb, float beta, float *C, int64_t ldc, int num_moduli,
                      int scaling_mode, void *stream)
{
    return blas_entry(1, layout, transa, transb, m, n, k, (double)alpha, A, lda, B, ldb, (double)beta, C, ldc, num_moduli,
                      scaling_mode, static_cast<cudaStream_t>(stream));
}

const char *ozaki2_status_string(int status)
{
    // names in the numbering of ozaki2_dgemm / ozaki2_dgemm_host (other entry points shift them as their
    // headers say; the number is always the position in the prototype that was called)
    static const char *arg_names[] = { "",      "m",   "n",    "k", "alpha",      "A",           "lda",   "B",
                                       "ldb",   "beta", "C",   "ldc", "num_moduli", "scaling_mode", "stream / device_scratch" };
    static thread_local char buf[128];
    if (status == 0) return "success";
    if (status == OZAKI2_ERR_WORKSPACE) return "workspace missing or too small (ozaki2_set_workspace)";
    if (status == OZAKI2_ERR_DEVICE) return "current device is not sm_100 (B200)";
    if (status == OZAKI2_ERR_NOALLOC_LIMIT)
        return "more rows than the built-in scratch of ozaki2_row_exponents_noalloc holds (OZAKI2_NOALLOC_MAX_ROWS = 65536): split the rows";
    if (status < 0 && status >= -14) {
        snprintf(buf, sizeof buf, "invalid argument %d (ozaki2_dgemm numbering: %s)", -status, arg_names[-status]);
        return buf;
    }
    if (status < 0 && status > -100) {
        snprintf(buf, sizeof buf, "invalid argument %d", -status);
        return buf;
    }
    if (status > 0) return cudaGetErrorString(static_cast<cudaError_t>(status));
    return "unknown status";
}

int ozaki2_get_constants(int num_moduli, int32_t *p, int32_t *q, uint64_t *P_words, uint64_t *w_words, float *Pprop,
                         float *Pfast, float *delta)
{
    if (num_moduli < OZAKI2_MIN_MODULI || num_moduli > OZAKI2_MAX_MODULI) return -1;
    HostConsts &H = host_consts();
    const int N = num_moduli;
    auto pack = [](const Big &b, uint64_t *dst) {
        for (int t = 0; t < 4; t++) {
            uint64_t lo = 2 * t < (int)b.size() ? b[2 * t] : 0, hi = 2 * t + 1 < (int)b.size() ? b[2 * t + 1] : 0;
            dst[t] = lo | (hi << 32);
        }
    };
    for (int l = 0; l < N; l++) {
        if (p) p[l] = kModuli[l];
        if (q) q[l] = H.q[N][l];
        if (w_words) pack(H.w[N][l], w_words + 4 * l);
    }
    if (P_words) pack(H.P[N], P_words);
    if (Pprop) *Pprop = H.tab.crt[N].Pprop;
    if (Pfast) *Pfast = H.tab.crt[N].Pfast;
    if (delta) *delta = H.tab.crt[N].delta;
    return 0;
}

int ozaki2_debug_log2f(const float *x, float *y, int64_t count, void *stream)
{
    DeviceState *dev = nullptr;
    int rc = ensure_device(&dev);
    if (rc) return rc;
    if (count < 0) return -3;
    return oz2_launch_log2f(x, y, count, static_cast<cudaStream_t>(stream));
}

int ozaki2_debug_mod_p(int modulus_index, const int32_t *in, uint8_t *out, int64_t count, void *stream)
{
    DeviceState *dev = nullptr;
    int rc = ensure_device(&dev);
    if (rc) return rc;
    if (modulus_index < 0 || modulus_index >= OZ2_MAX_MODULI) return -1;
    if (count < 0) return -4;
    return oz2_launch_mod_p(modulus_index, in, out, count, static_cast<cudaStream_t>(stream));
}

int ozaki2_debug_residue_gemm(int num_moduli, int64_t m, int64_t n, int64_t k, const int8_t *resA, const int8_t *resB,
                              uint8_t *U, int use_tensor_cores, void *stream)
{
    DeviceState *dev = nullptr;
    int rc = ensure_device(&dev);
    if (rc) return rc;
    if (num_moduli < 1 || num_moduli > OZAKI2_MAX_MODULI) return -1;
    if (m < 0) return -2;
    if (n < 0) return -3;
    if (k <= 0 || k % 128 != 0 || k > OZAKI2_MAX_K) return -4;      // canonical planes are used in place: pitch = k
    if (m % 16 != 0) return -2;                                     // U pitch = m
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (use_tensor_cores < 0 || use_tensor_cores > 4) return -8;
    if (use_tensor_cores) {
        // 1: one CTA per tile, 2: CTA pairs (the ozaki2_dgemm path), 3 / 4: the kernels of 1 / 2 without their epilogue
        const int variant = use_tensor_cores == 2 ? OZ2_GEMM_PAIR : use_tensor_cores == 3 ? OZ2_GEMM_MMA_ONLY
                            : use_tensor_cores == 4 ? OZ2_GEMM_PAIR_MMA_ONLY : OZ2_GEMM_PATH;
        return oz2_launch_gemm_tc(variant, num_moduli, 0, m, n, k, resA, resB, k, U, m, nullptr, nullptr, st);
    }
    return oz2_launch_gemm_check(num_moduli, m, n, k, resA, resB, k, U, m, st);
}

size_t ozaki2_zgemm_workspace_bytes(int64_t m, int64_t n, int64_t k, int num_moduli, int scaling_mode)
{
    return complex_workspace_bytes(8, m, n, k, num_moduli, scaling_mode);
}
size_t ozaki2_cgemm_workspace_bytes(int64_t m, int64_t n, int64_t k, int num_moduli, int scaling_mode)
{
    return complex_workspace_bytes(4, m, n, k, num_moduli, scaling_mode);
}

int ozaki2_zgemm(int64_t m, int64_t n, int64_t k, double alpha_re, double alpha_im, const double *A, int64_t lda,
                 const double *B, int64_t ldb, double beta_re, double beta_im, double *C, int64_t ldc, int num_moduli,
                 int scaling_mode, void *stream)
{
    return complex_entry<double>(m, n, k, alpha_re, alpha_im, A, lda, B, ldb, beta_re, beta_im, C, ldc, num_moduli, scaling_mode, stream);
}

int ozaki2_cgemm(int64_t m, int64_t n, int64_t k, float alpha_re, float alpha_im, const float *A, int64_t lda,
                 const float *B, int64_t ldb, float beta_re, float beta_im, float *C, int64_t ldc, int num_moduli,
                 int scaling_mode, void *stream)
{
    return complex_entry<float>(m, n, k, alpha_re, alpha_im, A, lda, B, ldb, beta_re, beta_im, C, ldc, num_moduli, scaling_mode, stream);
}

int ozaki2_debug_crt(int num_moduli, int64_t m, int64_t n, const uint8_t *U, const int32_t *e, const int32_t *f, double alpha,
                     double beta, void *C, int64_t ldc, uint64_t *Cpp, int is_f32, void *stream)
{
    DeviceState *dev = nullptr;
    int rc = ensure_device(&dev);
    if (rc) return rc;
    if (num_moduli < OZAKI2_MIN_MODULI || num_moduli > OZAKI2_MAX_MODULI) return -1;
    if (m < 0 || m % 16 != 0) return -2;                            // the planes are used in place: pitch = m
    if (n < 0) return -3;
    if (m == 0 || n == 0) return 0;
    if (!U) return -4;
    if (!e) return -5;
    if (!f) return -6;
    if (!C) return -9;
    if (ldc < m) return -10;
    return oz2_launch_crt(num_moduli, is_f32 ? 1 : 0, m, n, U, m, e, f, alpha, beta, C, ldc, Cpp, static_cast<cudaStream_t>(stream));
}

// S1 for the rows of A with the row statistics in the library's own static device array (oz2_scale.cu): for callers
// that have no way of allocating a workspace.  Checks first, so that an oversized problem touches nothing.
int ozaki2_row_exponents_noalloc(int64_t m, int64_t k, const double *A, int64_t lda, int num_moduli, int scaling_mode,
                                 int32_t *e, void *stream)
{
    static_assert(OZAKI2_NOALLOC_MAX_ROWS == OZ2_NOALLOC_MAX_ROWS, "header and kernel source disagree on the limit");
    if (m < 0) return -1;
    if (m > OZAKI2_NOALLOC_MAX_ROWS) return OZAKI2_ERR_NOALLOC_LIMIT;
    if (k < 0 || k > OZAKI2_MAX_K) return -2;
    if (m > 0 && k > 0 && !A) return -3;
    if (lda < (m > 1 ? m : 1)) return -4;
    if (num_moduli < OZAKI2_MIN_MODULI || num_moduli > OZAKI2_MAX_MODULI) return -5;
    if (scaling_mode != OZAKI2_MODE_FAST && scaling_mode != OZAKI2_MODE_PROP) return -6;
    if (m > 0 && !e) return -7;
    if (m == 0) return 0;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    DeviceState *dev = nullptr;
    int rc = ensure_device(&dev);
    if (rc) return rc;
    if (k == 0) {                                                   // empty rows are zero rows: exponent 0 (reading R4)
        OZ2_CUDA_TRY(cudaMemsetAsync(e, 0, sizeof(int32_t) * (size_t)m, st));
        return 0;
    }
    return oz2_launch_scale_rows_noalloc(scaling_mode, num_moduli, m, k, A, lda, e, st);
}

uint64_t ozaki2_kernel_launches(void) { return g_launches.load(std::memory_order_relaxed); }

const char *ozaki2_version(void) { return "ozaki2 0.1 sm_100a tcgen05.kind::i8 (arxiv/paper_2606_29129)"; }

} // extern "C"
