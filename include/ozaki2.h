/*
 * ozaki2.h -- C ABI of the B200-native Ozaki-scheme-II DGEMM library (libozaki2.so).
 *
 * The library emulates C = alpha * A B + beta * C in FP64 on the INT8 tensor cores of one
 * B200 (sm_100a), following "Improved Scaling for Fast Mode of Ozaki Scheme II"
 * (PAPER.md, cited as P:<line>): Steps 1-4 of section 2.2 with the three ways
 * of choosing the scaling vectors mu, nu of section 2.3 / section 4.
 *
 * Conventions for every entry point
 *   - plain pointers and sizes only; "device pointer" = memory of the current CUDA device,
 *     "host pointer" = ordinary host memory.  Nothing is allocated or freed for the caller.
 *   - matrices are column-major (BLAS "NN"): A is m x k with leading dimension lda >= max(1,m),
 *     B is k x n with ldb >= max(1,k), C is m x n with ldc >= max(1,m).
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Calls
 *     that take a stream only enqueue work: no host synchronisation, no allocation.
 *   - return value: 0 on success; -i if the i-th argument (1-based, as written in the
 *     prototype) is invalid; OZAKI2_ERR_WORKSPACE if the workspace is missing or too small;
 *     OZAKI2_ERR_DEVICE if the device is not sm_100; a positive value is a cudaError_t from a
 *     launch or copy.  Nothing throws across this boundary.
 *   - non-finite inputs are not detected: a row of A / column of B holding Inf or NaN gives
 *     unspecified values in that row / column of C (never a hang or a fault).
 */
#ifndef OZAKI2_H
#define OZAKI2_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* scaling_mode */
#define OZAKI2_MODE_ACCURATE 0 /* accurate mode: auxiliary INT8 GEMM, eq. (4)-(9)      */
#define OZAKI2_MODE_FAST 1     /* original fast mode: Algorithm 1, eq. (11)(12)        */
#define OZAKI2_MODE_PROP 2     /* revised fast mode: Algorithm 2, eq. (17)(18)         */

#define OZAKI2_MIN_MODULI 2
#define OZAKI2_MAX_MODULI 20           /* prefix of eq. (14)                           */
#define OZAKI2_K_BLOCK (1 << 17)       /* INT32 accumulator bound: longer k is blocked      */
#define OZAKI2_MAX_K (1 << 22)         /* blocked products up to here (sum of squares in 64 bits)  */
#define OZAKI2_MAX_K_ACCURATE (1 << 18) /* accurate mode: the auxiliary product 2^12 k fits INT32  */

#define OZAKI2_ERR_WORKSPACE (-100)
#define OZAKI2_ERR_DEVICE (-101)

/*
 * The hot path.  C := alpha * (A B)~ + beta * C, where (A B)~ is the Ozaki-II emulation with
 * `num_moduli` moduli (the first num_moduli of eq. (14)) and scaling mode `scaling_mode`:
 *   S1  mu_i = 2^e_i, nu_j = 2^f_j from row / column statistics
 *   S2  A' = trunc(diag(mu) A), B' = trunc(B diag(nu)); INT8 residues rmod(., p_l)
 *   S3  U_l = (rmod(A',p_l) rmod(B',p_l)) mod p_l on the INT8 tensor cores, l = 1..N    (eq. 2)
 *   S4  C'' = rmod(sum_l P_l q_l U_l, P)                                          (eq. 2, 3)
 *   S5  C = diag(mu)^-1 C'' diag(nu)^-1, then alpha / beta
 * A, B, C: device pointers, 8-byte aligned; C must not overlap A or B.  C is read only if
 * beta != 0.  alpha, beta by value.  Quick returns: m == 0 or n == 0 does nothing; k == 0 or
 * alpha == 0 gives C := beta * C (zeros if beta == 0).  k <= OZAKI2_MAX_K (OZAKI2_MAX_K_ACCURATE in
 * accurate mode); beyond OZAKI2_K_BLOCK the residue products are computed in blocks of 2^17 and summed mod p_l
 * (P:113).
 * Needs a workspace of ozaki2_workspace_bytes(m, n, k, num_moduli, scaling_mode) bytes
 * registered with ozaki2_set_workspace for the current device.  Asynchronous on `stream`.  After the first call
 * on a device (which uploads the constant tables) the call only enqueues kernels and memsets on `stream` and can
 * be captured into a CUDA graph.
 */
int ozaki2_dgemm(int64_t m, int64_t n, int64_t k, double alpha, const double *A, int64_t lda,
                 const double *B, int64_t ldb, double beta, double *C, int64_t ldc,
                 int num_moduli, int scaling_mode, void *stream);

/*
 * Transposed operands (the paper states C = A B only): C := alpha op(A) op(B) + beta C with
 * op(X) = X (trans = 0) or X^T (trans = 1).  A is stored m x k (transa = 0) or k x m (transa = 1), B is stored
 * k x n or n x k, column-major, lda / ldb >= the stored row count.  Same results as ozaki2_dgemm on the
 * materialised op(A), op(B), bit for bit.  Errors: -1 / -2 for a bad flag, then -(i + 2) for argument i of
 * ozaki2_dgemm.
 */
int ozaki2_dgemm_t(int transa, int transb, int64_t m, int64_t n, int64_t k, double alpha, const double *A,
                   int64_t lda, const double *B, int64_t ldb, double beta, double *C, int64_t ldc,
                   int num_moduli, int scaling_mode, void *stream);

/*
 * The full BLAS shape (the paper states C = A B only).  `layout`: 'C' column-major or 'R'
 * row-major (any case; the CBLAS enums 102 / 101 are accepted too).  `transa`, `transb`: 'N', 'T' or 'C' (any case;
 * 'C' = 'T' for real matrices; CBLAS 111 / 112 / 113).  Column-major: exactly ozaki2_dgemm_t.  Row-major: A is stored
 * m x k (transa = 'N', lda >= k) or k x m ('T', lda >= m), B is k x n (ldb >= n) or n x k (ldb >= k), C is m x n with
 * ldc >= n, all with the column index fastest.  A row-major problem is run as the column-major problem
 * C^T = op(B)^T op(A)^T on the same memory; the scaled vectors (rows of op(A), columns of op(B)) are the same in both
 * views, so the result equals ozaki2_dgemm on the logical matrices bit for bit.  Errors: -1 / -2 / -3 for a bad flag,
 * then -(i + 3) for argument i of ozaki2_dgemm (of the caller's A, B: the internal operand swap is undone).
 */
int ozaki2_dgemm_blas(int layout, int transa, int transb, int64_t m, int64_t n, int64_t k, double alpha, const double *A,
                      int64_t lda, const double *B, int64_t ldb, double beta, double *C, int64_t ldc, int num_moduli,
                      int scaling_mode, void *stream);
/* Workspace of an ozaki2_dgemm_blas / ozaki2_sgemm_blas call with this `layout` (same flag values; 0 for an invalid problem):
 * ozaki2_workspace_bytes(m, n, k, ...) for column-major and ozaki2_workspace_bytes(n, m, k, ...) for row-major, because a
 * row-major call runs internally with m and n exchanged (with m = 300, n = 1 the row-major call needs the larger figure). */
size_t ozaki2_blas_workspace_bytes(int layout, int64_t m, int64_t n, int64_t k, int num_moduli, int scaling_mode);

/*
 * SGEMM variant (Fig. 6): A, B, C are FP32 (4-byte aligned device pointers, same
 * column-major conventions).  Every FP32 input is an FP64 number, so S1-S4 are the steps above on
 * the promoted inputs; S5 rounds the exact integer once to FP32, C = RN_32(C'' 2^-(e_i+f_j)), and
 * alpha / beta are applied in FP32 (t = alpha C; out = beta == 0 ? t : fmaf(beta, C_in, t)).  Same
 * workspace, quick returns and error codes as ozaki2_dgemm; the paper uses 3..12 moduli here.
 */
int ozaki2_sgemm(int64_t m, int64_t n, int64_t k, float alpha, const float *A, int64_t lda,
                 const float *B, int64_t ldb, float beta, float *C, int64_t ldc,
                 int num_moduli, int scaling_mode, void *stream);

/* The transposed-operand and full-BLAS entry points of the SGEMM variant (same conventions as the FP64 ones). */
int ozaki2_sgemm_t(int transa, int transb, int64_t m, int64_t n, int64_t k, float alpha, const float *A, int64_t lda,
                   const float *B, int64_t ldb, float beta, float *C, int64_t ldc, int num_moduli, int scaling_mode,
                   void *stream);
int ozaki2_sgemm_blas(int layout, int transa, int transb, int64_t m, int64_t n, int64_t k, float alpha, const float *A,
                      int64_t lda, const float *B, int64_t ldb, float beta, float *C, int64_t ldc, int num_moduli,
                      int scaling_mode, void *stream);

/*
 * Complex variant (named as future work at P:58, P:444 without formulas -- reading in DESIGN.md 8b #4):
 * C := alpha A B + beta C for interleaved complex FP64 matrices (re, im pairs; column-major; lda, ldb, ldc in complex
 * elements; 16-byte aligned device pointers), computed as ozaki2_dgemm on the real embedding
 * [C_r; C_i] = [[A_r, -A_i], [A_i, A_r]] [B_r; B_i]  (a (2m x 2k)(2k x n) product: one scaling exponent per complex row
 * of A / column of B, condition (1) holds for both parts), then out = alpha c + beta C in plain complex arithmetic with
 * every product and sum rounded on its own (alpha == 1, beta == 0 and beta == 1 are not multiplied: beta == 0 overwrites,
 * beta == 1 adds C as it is, and with k == 0 or alpha == 0 leaves C untouched, as the real entry points do).  The
 * embedded operands are materialised in the workspace: register ozaki2_zgemm_workspace_bytes(...) bytes with
 * ozaki2_set_workspace.  2k <= OZAKI2_MAX_K (OZAKI2_MAX_K_ACCURATE in accurate mode).  Errors: -i for argument i.
 */
int ozaki2_zgemm(int64_t m, int64_t n, int64_t k, double alpha_re, double alpha_im, const double *A, int64_t lda,
                 const double *B, int64_t ldb, double beta_re, double beta_im, double *C, int64_t ldc,
                 int num_moduli, int scaling_mode, void *stream);
size_t ozaki2_zgemm_workspace_bytes(int64_t m, int64_t n, int64_t k, int num_moduli, int scaling_mode);

/*
 * The same for interleaved complex FP32 matrices (8-byte aligned device pointers): ozaki2_sgemm on the real embedding of the
 * FP32 parts (one rounding RN_32 of the exact integer for each of c_r, c_i; P:375 for the moduli counts), then the tail
 * out = alpha c + beta C with every product and sum rounded to FP32 on its own.  Workspace: ozaki2_cgemm_workspace_bytes.
 */
int ozaki2_cgemm(int64_t m, int64_t n, int64_t k, float alpha_re, float alpha_im, const float *A, int64_t lda,
                 const float *B, int64_t ldb, float beta_re, float beta_im, float *C, int64_t ldc,
                 int num_moduli, int scaling_mode, void *stream);
size_t ozaki2_cgemm_workspace_bytes(int64_t m, int64_t n, int64_t k, int num_moduli, int scaling_mode);

/* Bytes of device workspace ozaki2_dgemm / ozaki2_sgemm (and their _t, _ws, _stages forms) need for this problem (0 for an
 * invalid one).  The figure is NOT symmetric in m and n. */
size_t ozaki2_workspace_bytes(int64_t m, int64_t n, int64_t k, int num_moduli, int scaling_mode);

/*
 * Register a caller-owned device buffer (256-byte aligned) as the workspace of the current
 * device; it must stay valid until replaced.  (NULL, 0) unregisters.  Not stream ordered: do
 * not replace it while calls that use it are in flight.  All calls on a device share this one
 * workspace, so concurrent calls must be ordered with respect to each other (same stream, or
 * events); calls on different devices are independent.
 */
int ozaki2_set_workspace(void *device_ptr, size_t bytes);

/*
 * ozaki2_dgemm / ozaki2_sgemm with the workspace of THIS call passed in (device pointer, 256-byte aligned, at least
 * ozaki2_workspace_bytes(m, n, k, num_moduli, scaling_mode) bytes; it must stay valid until the call's work on `stream`
 * has finished): calls that use different workspaces are independent and may run concurrently on different streams or from
 * different host threads.  The registered workspace of the device is not touched.  A missing, misaligned or too small
 * workspace returns -14 (its argument number).  Everything else as ozaki2_dgemm / ozaki2_sgemm.
 */
int ozaki2_dgemm_ws(int64_t m, int64_t n, int64_t k, double alpha, const double *A, int64_t lda, const double *B,
                    int64_t ldb, double beta, double *C, int64_t ldc, int num_moduli, int scaling_mode,
                    void *workspace, size_t workspace_bytes, void *stream);
int ozaki2_sgemm_ws(int64_t m, int64_t n, int64_t k, float alpha, const float *A, int64_t lda, const float *B,
                    int64_t ldb, float beta, float *C, int64_t ldc, int num_moduli, int scaling_mode,
                    void *workspace, size_t workspace_bytes, void *stream);

/*
 * The same call with HOST buffers: copies A and B to the device, runs ozaki2_dgemm, copies C
 * back (and C in first if beta != 0), then synchronises `stream`.  For the two fast modes and
 * n >= 512 the work is cut into column panels of B / C: the kernels stay on `stream`, the copies
 * run on two library-owned streams ordered after `stream` by events, so that the H2D copy of the
 * next panel and the D2H copy of the previous one overlap the kernels (same results bit for bit:
 * e_i depends on row i of A only, f_j on column j of B only).
 * `device_scratch` is a caller-owned device buffer of at least
 * ozaki2_host_scratch_bytes(m, n, k) bytes that receives the device copies of A, B, C (the FP32 variant needs
 * half of it); a missing or short buffer is error -14.  Host buffers should be page-locked for the copies to run
 * at link speed.  The call returns only after every copy it enqueued has finished, also when it returns an error.
 */
int ozaki2_dgemm_host(int64_t m, int64_t n, int64_t k, double alpha, const double *A_host, int64_t lda,
                      const double *B_host, int64_t ldb, double beta, double *C_host, int64_t ldc,
                      int num_moduli, int scaling_mode, void *device_scratch, size_t scratch_bytes,
                      void *stream);
int ozaki2_sgemm_host(int64_t m, int64_t n, int64_t k, float alpha, const float *A_host, int64_t lda,
                      const float *B_host, int64_t ldb, float beta, float *C_host, int64_t ldc,
                      int num_moduli, int scaling_mode, void *device_scratch, size_t scratch_bytes,
                      void *stream);
size_t ozaki2_host_scratch_bytes(int64_t m, int64_t n, int64_t k);

/*
 * S1 for the rows of A without any memory from the caller beyond the input and the output: e[i] = log2 mu_i of
 * Algorithm 1 (OZAKI2_MODE_FAST) or Algorithm 2 (OZAKI2_MODE_PROP) for the m rows of the
 * column-major m x k matrix A -- the same kernels, and therefore the same integers, as the `e` that ozaki2_dgemm
 * computes for its A.  (Accurate mode needs B and an auxiliary product; it is rejected with -6.)
 *
 * Who this is for.  Every other compute call of this library needs a workspace, which somebody has to cudaMalloc.
 * Some callers may not, or cannot: a plug-in running under a host application that took all of the device memory
 * for its own pool at start-up (a further cudaMalloc fails there, and the host's pool is not ours to carve); code
 * in a latency-critical loop, where cudaMalloc / cudaFree stall the whole device, not one stream; a component
 * whose rules simply forbid driver allocations after initialisation.  For them the row statistics of the two
 * streaming passes (max |a_ih| and the integer sum of squares, 16 bytes per row) live in an array that is part of
 * the library image itself: OZAKI2_NOALLOC_MAX_ROWS rows, 1 MiB, present on every GPU that loads the library from
 * the moment it is loaded until the process exits, whether this call is used or not.  The call runs no cudaMalloc,
 * cudaFree or any routine that allocates; it enqueues one memset and three kernels on `stream`.
 *
 * Limits and rules.
 *   - m <= OZAKI2_NOALLOC_MAX_ROWS; a larger m returns OZAKI2_ERR_NOALLOC_LIMIT and enqueues nothing (split the rows:
 *     e[i] depends on row i only).  k <= OZAKI2_MAX_K.  k == 0 gives e[i] = 0.
 *   - The first call on each device looks up where that device keeps the array (and, like every entry point, uploads
 *     the constant tables if no other call has yet).  Make that first call during initialisation, with the device
 *     current and outside any stream capture.
 *   - There is ONE array per device and every call uses it.  Each call zeroes the part it needs on `stream` before
 *     its kernels, so what an earlier call left behind is harmless -- but two calls whose GPU work can overlap
 *     (different streams without an event between them, or different host threads on different streams) read and
 *     write the same statistics and both get wrong exponents.  Order them: one stream, or events.
 * A: device pointer, lda >= max(1, m); e: device pointer to m int32.  Errors: -i for argument i of this prototype.
 */
#define OZAKI2_NOALLOC_MAX_ROWS 65536
#define OZAKI2_ERR_NOALLOC_LIMIT (-102)
int ozaki2_row_exponents_noalloc(int64_t m, int64_t k, const double *A, int64_t lda, int num_moduli, int scaling_mode,
                                 int32_t *e, void *stream);

/*
 * Environment.  The library reads two variables, once, when it is first used; neither changes a result:
 *   OZAKI2_PDL=0        launch every kernel the plain way instead of chaining the kernels of a call by programmatic
 *                       dependent launch (a diagnostic switch: profilers and sanitizers see ordinary launches)
 *   OZAKI2_GEMM=single  run S3 on the one-CTA-per-tile kernel instead of CTA pairs
 * Everything else is an argument.
 */

/* Text for a return value of this library. */
const char *ozaki2_status_string(int status);

/* ------------------------------------------------------------------------------------------
 * Parity and profiling surface.  ozaki2_dgemm_stages runs exactly the kernels of ozaki2_dgemm
 * and, in addition, copies the intermediate results of each stage into the caller's device
 * buffers in CANONICAL layouts (independent of the internal pitches).  Every pointer may be
 * NULL (= not wanted).
 * ---------------------------------------------------------------------------------------- */
typedef struct ozaki2_stage_outputs {
    int32_t *e;          /* [m]        log2 mu_i                                              */
    int32_t *f;          /* [n]        log2 nu_j                                              */
    int32_t *rowmax;     /* [m]        max_j cbar_ij, accurate mode only          */
    int32_t *colmax;     /* [n]        max_i cbar_ij, accurate mode only                      */
    int8_t *resA;        /* [N][m][k]  symmetric INT8 residues of A', k fastest               */
    int8_t *resB;        /* [N][n][k]  symmetric INT8 residues of B', k fastest               */
    uint8_t *U;          /* [N][n][m]  (resA_l resB_l^T) mod p_l in [0,p_l), m fastest        */
    uint64_t *Cpp;       /* [n][m][4]  C'' as 256-bit two's-complement words, little-endian   */
    float *stage_ms;     /* HOST pointer, [5]: elapsed ms of S1, S2, S3, S4+S5, total; filling
                            it synchronises the stream (profiling only)                       */
    void **stage_events; /* HOST array of 5 caller-owned cudaEvent_t (timing enabled): recorded on
                            `stream` before S1 and after S1, S2, S3, S4+S5.  No synchronisation:
                            the caller reads them with cudaEventElapsedTime after its own sync  */
} ozaki2_stage_outputs;

int ozaki2_dgemm_stages(int64_t m, int64_t n, int64_t k, double alpha, const double *A, int64_t lda,
                        const double *B, int64_t ldb, double beta, double *C, int64_t ldc,
                        int num_moduli, int scaling_mode, void *stream, const ozaki2_stage_outputs *out);

/* ozaki2_dgemm_stages for the SGEMM variant (same outputs; C'' is the same integer as in the FP64 path). */
int ozaki2_sgemm_stages(int64_t m, int64_t n, int64_t k, float alpha, const float *A, int64_t lda, const float *B,
                        int64_t ldb, float beta, float *C, int64_t ldc, int num_moduli, int scaling_mode,
                        void *stream, const ozaki2_stage_outputs *out);

/*
 * Constants of Step 1 for `num_moduli` moduli, written to HOST arrays (any may be NULL):
 * p[N], q[N] (q_l = P_l^-1 mod p_l), P_words[4] and w_words[N][4] (w_l = P_l q_l,
 * eq. (2)) as little-endian 64-bit words, and the FP32 constants P'_prop = P'_accu
 * (P:141-143), P'_fast, delta (eq. (6)).
 */
int ozaki2_get_constants(int num_moduli, int32_t *p, int32_t *q, uint64_t *P_words, uint64_t *w_words,
                         float *Pprop, float *Pfast, float *delta);

/* y[t] = LOG2F(x[t]) for x[t] in [1,2]: the library's stand-in for __log2f (R3),
 * evaluated on the device.  x, y: device pointers. */
int ozaki2_debug_log2f(const float *x, float *y, int64_t count, void *stream);

/* out[t] = in[t] mod p_l in [0,p_l) for any INT32 in[t], computed by the same routine as the
 * epilogue of the residue GEMM.  in, out: device pointers. */
int ozaki2_debug_mod_p(int modulus_index, const int32_t *in, uint8_t *out, int64_t count, void *stream);

/* One INT8 product resA_l resB_l^T mod p_l for canonical planes (same layouts as above) on a
 * tensor-core kernel -- use_tensor_cores = 2: the cta_group::2 kernel, CTA pairs on 256 x 256 tiles,
 * what ozaki2_dgemm runs (for m > 128 and k <= OZAKI2_K_BLOCK); 1: one CTA per 128 x 256 tile, what
 * it runs otherwise and the measured alternative; 3 / 4: the kernels of 1 / 2 with the epilogue
 * reduced to handing the accumulator back, U untouched (the INT8 ceiling of each loop that bench.py
 * measures) -- or on a plain CUDA-core check kernel (0) that ozaki2_dgemm never uses.  k must be a
 * multiple of 128 and m of 16 (the planes are used in place).  None needs a workspace. */
int ozaki2_debug_residue_gemm(int num_moduli, int64_t m, int64_t n, int64_t k, const int8_t *resA,
                              const int8_t *resB, uint8_t *U, int use_tensor_cores, void *stream);

/* S4 + S5 on caller-made residue planes (eq. (2)(3); Step 4): runs the CRT kernel of
 * ozaki2_dgemm on U [N][n][m] (uint8, m fastest, m a multiple of 16; U_l < p_l), exponents e[m], f[n] (device),
 * and writes C := alpha RN(C'') 2^-(e_i+f_j) + beta C (FP64, or FP32 if is_f32) with leading dimension ldc.
 * Cpp == NULL: the production code path (branch-free common case, exact routine for the rare ones);
 * Cpp != NULL ([n][m][4] u64): the exact routine for every element, which also stores C''.
 * alpha, beta are rounded to FP32 when is_f32.  Errors: -i for argument i. */
int ozaki2_debug_crt(int num_moduli, int64_t m, int64_t n, const uint8_t *U, const int32_t *e, const int32_t *f,
                     double alpha, double beta, void *C, int64_t ldc, uint64_t *Cpp, int is_f32, void *stream);

/* Number of kernels this library has launched in this process so far (all devices, all entry
 * points; memsets and copies are not counted). */
uint64_t ozaki2_kernel_launches(void);

/* Library build information: "ozaki2 <version> sm_100a ..." */
const char *ozaki2_version(void);

#ifdef __cplusplus
}
#endif
#endif /* OZAKI2_H */
