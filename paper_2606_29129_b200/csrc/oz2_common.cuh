// oz2_common.cuh -- shared declarations of the libozaki2 CUDA sources (product code; the
// CPU oracle under oracle/ shares nothing with this tree).
//
// Notation follows PAPER.md (P:<line>): moduli p_l, P = prod p_l, mu_i = 2^e_i, nu_j = 2^f_j,
// A' = trunc(diag(mu) A), residues rmod(A', p_l), U_l, C'', C.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define OZ2_MAX_MODULI 20
#define OZ2_MAX_WORDS 6          // 32-bit words of a CRT weight: log2 P <= 155.4  ->  5 words (+1 for sums)

// eq. (14).  Index l = 0 is p = 256.
#define OZ2_MODULI_LIST { 256, 255, 253, 251, 247, 241, 239, 233, 229, 227, 223, 217, 211, 199, 197, 193, 191, 181, 179, 173 }

// ----- per-modulus table (independent of N) ---------------------------------------------------
struct Oz2ModTab {
    uint32_t p;            // modulus
    uint32_t magic;        // floor(2^32 / p) + 1 : floor(x / p) = umulhi(x, magic) for x < 2^24 (x * p_err < 2^32)
    uint32_t half;         // (p - 1) / 2
    uint32_t conv_bias;    // multiple of p, >= largest |signed dot| of the conversion kernel
    uint32_t wb[3];        // byte weights 256^(4t+b) mod p, b = 0..3 packed little-endian, t = 0..2
    uint32_t w16;          // 2^16 mod p                           (epilogue: R = hi * 2^16 + lo)
    uint32_t epi_bias;     // multiple of p, >= 2^15 * w16
    uint32_t pad[3];
};

// ----- per-N table -----------------------------------------------------------------------------
struct Oz2CrtTab {
    uint32_t w[OZ2_MAX_MODULI][OZ2_MAX_WORDS];   // w_l = P_l q_l (< P), little-endian 32-bit words
    uint32_t P[OZ2_MAX_WORDS];                   // P
    uint32_t Phalf[OZ2_MAX_WORDS];               // P / 2 (P is even: 256 | P)
    double invP;                                 // RN(1 / P)
    int32_t nw;                                  // number of 32-bit words of P
    float Pprop, Pfast, delta;                   // P:326-328 (= P'_accu P:141-143), eq. (6)
};

struct Oz2HostTables {
    Oz2ModTab mod[OZ2_MAX_MODULI];
    Oz2CrtTab crt[OZ2_MAX_MODULI + 1];           // index N
};

// internal pitches: residue planes are [l][row][kp] with kp = round_up(k, 128) bytes (zero padded),
// U planes are [l][j][mp] with mp = round_up(m, 16)
static inline __host__ __device__ int64_t oz2_round_up(int64_t x, int64_t q) { return (x + q - 1) / q * q; }

// launch helpers implemented by the kernel sources (all asynchronous on `st`)
int oz2_scale_upload_tables(const Oz2HostTables &t);
int oz2_convert_upload_tables(const Oz2HostTables &t);
int oz2_gemm_upload_tables(const Oz2HostTables &t);
int oz2_crt_upload_tables(const Oz2HostTables &t);

// S1: exponents for modes 1 and 2, and the mode-0 pieces.  stat buffers: amax[rows] (u64), ssq[rows] (u64)
// f32 != 0: the input matrices are FP32 (SGEMM variant); every element is promoted to FP64 exactly on load
int oz2_launch_scale_rows(int mode, int N, int f32, int64_t m, int64_t k, const void *A, int64_t lda,
                          unsigned long long *amaxA, unsigned long long *ssqA, int32_t *e, cudaStream_t st);
int oz2_launch_scale_cols(int mode, int N, int f32, int64_t n, int64_t k, const void *B, int64_t ldb, int32_t *f, cudaStream_t st);
int oz2_launch_scale_accu_side(int f32, int strided, int64_t cnt, int64_t k, const void *X, int64_t ldx,
                               unsigned long long *amax, int32_t *E, int8_t *bar, int64_t kp, cudaStream_t st);
int oz2_launch_scale_accu_finish(int N, int64_t m, int64_t n, const int32_t *EA, const int32_t *EB,
                                 const int32_t *rowmax, const int32_t *colmax, int32_t *e, int32_t *f, cudaStream_t st);
int oz2_launch_log2f(const float *x, float *y, int64_t count, cudaStream_t st);
// oz2_launch_scale_rows with amax / ssq in the library's own static device array (ozaki2_row_exponents_noalloc);
// m <= OZ2_NOALLOC_MAX_ROWS is the caller's check
#define OZ2_NOALLOC_MAX_ROWS 65536
int oz2_launch_scale_rows_noalloc(int mode, int N, int64_t m, int64_t k, const double *A, int64_t lda, int32_t *e, cudaStream_t st);

// S2: residues of op(X) for all N moduli in one pass.  planes: [N][rows][kp]
int oz2_launch_convert(int op, int N, int wide, int f32, int64_t rows, int64_t k, const void *X, int64_t ldx,
                       const int32_t *ex, int8_t *planes, int64_t kp, cudaStream_t st);

// S3: batched INT8 GEMM with mod-p epilogue (tcgen05).  nplanes GEMMs; modulus index of plane b is mod_base + b.
// U: [plane][n][mp].  If rowmax/colmax != NULL the epilogue keeps maxima instead (accurate mode).
// variant: OZ2_GEMM_PAIR (cta_group::2, CTA pairs on 256 x 256 tiles: what ozaki2_dgemm runs), OZ2_GEMM_PATH (one CTA per
// 128 x 256 tile: m <= 128, K-blocked products, OZAKI2_GEMM=single), OZ2_GEMM_MMA_ONLY / OZ2_GEMM_PAIR_MMA_ONLY (no epilogue)
enum { OZ2_GEMM_PATH = 0, OZ2_GEMM_PAIR = 1, OZ2_GEMM_MMA_ONLY = 2, OZ2_GEMM_PAIR_MMA_ONLY = 3 };
int oz2_launch_gemm_tc(int variant, int nplanes, int mod_base, int64_t m, int64_t n, int64_t k, const int8_t *RA,
                       const int8_t *RB, int64_t kp, uint8_t *U, int64_t mp, int32_t *rowmax, int32_t *colmax, cudaStream_t st);
int oz2_launch_gemm_check(int nplanes, int64_t m, int64_t n, int64_t k, const int8_t *RA, const int8_t *RB, int64_t kp,
                          uint8_t *U, int64_t mp, cudaStream_t st);
int oz2_launch_mod_p(int l, const int32_t *in, uint8_t *out, int64_t count, cudaStream_t st);

// S4 + S5: CRT, rmod P, RN to FP64, unscale, alpha / beta.  Cpp (optional): [n][m][4] u64 words.
// f32 != 0: C is FP32, the one rounding is RN_32, alpha / beta are applied in FP32
int oz2_launch_crt(int N, int f32, int64_t m, int64_t n, const uint8_t *U, int64_t mp, const int32_t *e, const int32_t *f,
                   double alpha, double beta, void *C, int64_t ldc, uint64_t *Cpp, cudaStream_t st);

// kernel-launch accounting behind ozaki2_kernel_launches()
void oz2_count_launches(int n);

// Programmatic dependent launch (PDL): every kernel of the path is launched with the programmatic-stream-serialization
// attribute, signals at its entry that its dependents may be scheduled (pdl_launch_dependents) and waits for its predecessor
// to complete and flush (pdl_wait) before it touches anything the predecessor wrote -- and in any case before it exits,
// which keeps the dependency transitive along the chain.  What runs before the wait (barrier initialisation, tensor-memory
// allocation, constant operand images) overlaps the predecessor's tail; at small sizes that is a good part of the call.
// Invariant for kernels that allocate tensor memory: they signal only AFTER tcgen05.alloc has returned and the CTA (pair) has
// synchronised on it.  Dependents become schedulable once every CTA of the predecessor has signalled, i.e. once all of them
// own their columns -- a dependent CTA that became resident earlier, took its columns and sat in pdl_wait could otherwise
// starve a predecessor CTA still blocked in tcgen05.alloc, which no time-out covers.
// OZAKI2_PDL=0 in the environment (read once) launches everything the plain way.
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
bool oz2_pdl_enabled();
template <typename... KArgs, typename... Args>
static inline cudaError_t oz2_launch(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args &&...args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = oz2_pdl_enabled() ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}
#endif

#define OZ2_CUDA_TRY(expr)                                   \
    do {                                                     \
        cudaError_t _e = (expr);                             \
        if (_e != cudaSuccess) return (int)_e;               \
    } while (0)
