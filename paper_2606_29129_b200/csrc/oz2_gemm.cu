// oz2_gemm.cu -- S3: the N residue products of eq. (2) ("the dominant cost is Step 3"),
//     U_l[j][i] = ( sum_h rA_l[i][h] * rB_l[j][h] ) mod p_l ,   l = 1..N,
// as ONE persistent tcgen05 kernel batched over the moduli, and -- same kernel, other epilogue -- the auxiliary
// product Cbar = Abar Bbar of accurate mode of which only row / column maxima are kept.
//
// sm_100a design (not the BLAS-call design of the paper's GH200 implementation):
//   * operands: INT8 planes, K-major, fetched by TMA (3-D tensor maps: k, row, plane) into a 4-stage ring of
//     SWIZZLE_128B shared-memory tiles (A 128 x 128 B, B 256 x 128 B per stage),
//   * math: tcgen05.mma.cta_group::1.kind::i8, M = 128, N = 256, K = 32 per instruction, issued by one thread;
//     INT32 accumulators live in tensor memory (2 x 256 columns, double buffered), they never touch HBM,
//   * epilogue: 4 warps read the accumulator with tcgen05.ld, reduce mod p_l and write one byte per element,
//     overlapping the MMAs of the next tile,
//   * persistent grid (one CTA per SM), static tile order: modulus-major, then groups of 32 M-tiles so that the
//     148 tiles in flight share A / B panels in L2.
// INT32 accumulation wraps (never saturates): with reading R6 that keeps k <= 2^17 exact for p = 256.
#include "oz2_common.cuh"
#include "oz2_tc.cuh"

namespace {

__constant__ Oz2ModTab c_mod[OZ2_MAX_MODULI];

constexpr int TILE_M = 128;
constexpr int TILE_N = 256;
constexpr int TILE_K = 128;                       // bytes = INT8 elements per stage (one 128B swizzle row)
constexpr int UMMA_K = 32;
constexpr int STAGES = 4;
constexpr int A_STAGE_BYTES = TILE_M * TILE_K;    // 16 KB
constexpr int B_STAGE_BYTES = TILE_N * TILE_K;    // 32 KB
constexpr int STAGE_BYTES = A_STAGE_BYTES + B_STAGE_BYTES;
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 1024 /*alignment slack*/ + 256 /*barriers*/;
constexpr int NUM_THREADS = 192;                  // warp 0: TMA, warp 1: MMA + TMEM alloc, warps 2..5: epilogue
constexpr int GROUP_M = 32;

// tcgen05 instruction descriptor (kind::i8): D = S32, A = B = signed 8 bit, both K-major, N = 256, M = 128
constexpr uint32_t IDESC = (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(TILE_N >> 3) << 17) |
                           ((uint32_t)(TILE_M >> 4) << 24);

// 32 lanes x 32 consecutive columns of 32-bit accumulators -> 32 registers per thread
__device__ __forceinline__ void tc_ld32(uint32_t taddr, uint32_t (&v)[32])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]),
          "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]),
          "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr)
        : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// shared-memory matrix descriptor: K-major, SWIZZLE_128B, rows of 128 B, 8-row groups 1024 B apart
__device__ __forceinline__ uint64_t make_smem_desc(uint32_t saddr)
{
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFFu) >> 4);         // start address
    d |= (uint64_t)(16u >> 4) << 16;                  // leading byte offset (unused for swizzled K-major)
    d |= (uint64_t)(1024u >> 4) << 32;                // stride byte offset between 8-row groups
    d |= 1ull << 46;                                  // descriptor version (sm_100)
    d |= 2ull << 61;                                  // SWIZZLE_128B
    return d;
}

// R mod p in [0, p) for any INT32 R (the GEMM epilogue and ozaki2_debug_mod_p share this routine):
// R = hi 2^16 + lo, hi in [-2^15, 2^15), lo in [0, 2^16);  y = hi w16 + lo + bias with bias = 0 (mod p) making
// y non-negative and y < 2^24 + 2^16, where umulhi(y, magic) is the exact quotient.
__device__ __forceinline__ uint32_t mod_p_i32(int32_t R, const Oz2ModTab &t)
{
    int32_t hi = R >> 16;
    uint32_t lo = (uint32_t)R & 0xFFFFu;
    uint32_t y = (uint32_t)(hi * (int32_t)t.w16 + (int32_t)t.epi_bias) + lo;
    uint32_t q = __umulhi(y, t.magic);
    return y - q * t.p;
}

struct TileCoord { int plane, m0, n0; };

__device__ __forceinline__ TileCoord decode_tile(int64_t t, int tiles_m, int tiles_n)
{
    const int64_t per_plane = (int64_t)tiles_m * tiles_n;
    TileCoord c;
    c.plane = (int)(t / per_plane);
    int rem = (int)(t - (int64_t)c.plane * per_plane);
    const int group_sz = GROUP_M * tiles_n;
    int g = rem / group_sz;
    int in_g = rem - g * group_sz;
    int gm = tiles_m - g * GROUP_M;
    if (gm > GROUP_M) gm = GROUP_M;
    int nt = in_g / gm;
    int mt = g * GROUP_M + (in_g - nt * gm);
    c.m0 = mt * TILE_M;
    c.n0 = nt * TILE_N;
    return c;
}

// MAXEPI = false: U[plane][j][mp] = acc mod p_(mod_base + plane);  true: rowmax / colmax of the accumulators
template <bool MAXEPI>
__global__ void __launch_bounds__(NUM_THREADS, 1)
k3_residue_gemm(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB, int nplanes,
                int mod_base, int m, int n, int num_kb, uint8_t *__restrict__ U, int64_t mp,
                int32_t *__restrict__ rowmax, int32_t *__restrict__ colmax)
{
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + STAGES * STAGE_BYTES);
    uint64_t *full = bars, *empty = bars + STAGES, *tfull = bars + 2 * STAGES, *tempty = bars + 2 * STAGES + 2;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(bars + 2 * STAGES + 4);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tiles_m = (m + TILE_M - 1) / TILE_M, tiles_n = (n + TILE_N - 1) / TILE_N;
    const int64_t total = (int64_t)nplanes * tiles_m * tiles_n;

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; s++) { mbar_init(full + s, 1); mbar_init(empty + s, 1); }
        for (int s = 0; s < 2; s++) { mbar_init(tfull + s, 1); mbar_init(tempty + s, 4); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&mapA) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&mapB) : "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        // ===================== TMA producer =====================
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (int64_t t = blockIdx.x; t < total; t += gridDim.x) {
                const TileCoord c = decode_tile(t, tiles_m, tiles_n);
                for (int kb = 0; kb < num_kb; kb++) {
                    mbar_wait(empty + stage, phase ^ 1u);
                    uint8_t *sa = smem + stage * STAGE_BYTES, *sb = sa + A_STAGE_BYTES;
                    mbar_expect_tx(full + stage, STAGE_BYTES);
                    tma_load_3d(&mapA, full + stage, sa, kb * TILE_K, c.m0, c.plane);
                    tma_load_3d(&mapB, full + stage, sb, kb * TILE_K, c.n0, c.plane);
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer =====================
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            int as = 0;
            uint32_t aphase = 0;
            for (int64_t t = blockIdx.x; t < total; t += gridDim.x) {
                mbar_wait(tempty + as, aphase ^ 1u);
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + (uint32_t)(as * TILE_N);
                for (int kb = 0; kb < num_kb; kb++) {
                    mbar_wait(full + stage, phase);
                    tc_fence_after();
                    const uint32_t sa = smem_u32(smem + stage * STAGE_BYTES), sb = sa + A_STAGE_BYTES;
                    const uint64_t adesc = make_smem_desc(sa), bdesc = make_smem_desc(sb);
#pragma unroll
                    for (int ks = 0; ks < TILE_K / UMMA_K; ks++)
                        tc_mma_i8(d_tmem, adesc + (uint64_t)(ks * UMMA_K / 16), bdesc + (uint64_t)(ks * UMMA_K / 16), IDESC,
                                  (uint32_t)((kb | ks) != 0));
                    tc_commit(empty + stage);                  // frees the smem stage when these MMAs retire
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
                tc_commit(tfull + as);                         // accumulator complete
                if (++as == 2) { as = 0; aphase ^= 1u; }
            }
        }
    } else {
        // ===================== epilogue: warps 2..5, TMEM lane quarter = warp % 4 =====================
        const int q = warp & 3;
        int as = 0;
        uint32_t aphase = 0;
        for (int64_t t = blockIdx.x; t < total; t += gridDim.x) {
            const TileCoord c = decode_tile(t, tiles_m, tiles_n);
            mbar_wait(tfull + as, aphase);
            tc_fence_after();
            const int i = c.m0 + q * 32 + lane;                // output row of this thread
            const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(as * TILE_N);
            if (!MAXEPI) {
                const int l = mod_base + c.plane;
                const Oz2ModTab tb = c_mod[l];
                uint8_t *out = U + ((int64_t)c.plane * n + c.n0) * mp + i;
#pragma unroll 1
                for (int cc = 0; cc < TILE_N / 32; cc++) {
                    uint32_t v[32];
                    tc_ld32(taddr + (uint32_t)(cc * 32), v);
                    if (i < m) {
#pragma unroll
                        for (int u = 0; u < 32; u++) {
                            const int j = c.n0 + cc * 32 + u;
                            uint32_t r = l == 0 ? (v[u] & 0xFFu) : mod_p_i32((int32_t)v[u], tb);
                            if (j < n) out[(int64_t)(cc * 32 + u) * mp] = (uint8_t)r;
                        }
                    }
                }
            } else {
                int rmax = 0;
#pragma unroll 1
                for (int cc = 0; cc < TILE_N / 32; cc++) {
                    uint32_t v[32];
                    tc_ld32(taddr + (uint32_t)(cc * 32), v);
#pragma unroll
                    for (int u = 0; u < 32; u++) {
                        const int j = c.n0 + cc * 32 + u;
                        int val = (i < m && j < n) ? (int)v[u] : 0;
                        rmax = max(rmax, val);
                        int cm = __reduce_max_sync(0xffffffffu, val);
                        if (lane == 0 && j < n && cm > 0) atomicMax(colmax + j, cm);
                    }
                }
                if (i < m && rmax > 0) atomicMax(rowmax + i, rmax);
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tempty + as);
            if (++as == 2) { as = 0; aphase ^= 1u; }
        }
    }
    __syncthreads();
    if (warp == 1) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
    }
}

// ---------------------------------------------------------------------------------------------
// plain CUDA-core check kernel (never on the ozaki2_dgemm path): one thread per (i, j), dp4a over k
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k3_check(int nplanes, int m, int n, int64_t kp, const int8_t *__restrict__ RA, const int8_t *__restrict__ RB,
         uint8_t *__restrict__ U, int64_t mp)
{
    const int i = blockIdx.x * 32 + (threadIdx.x & 31);
    const int j = blockIdx.y * 8 + (threadIdx.x >> 5);
    const int l = blockIdx.z;
    if (i >= m || j >= n) return;
    const int *a = reinterpret_cast<const int *>(RA + ((int64_t)l * m + i) * kp);
    const int *b = reinterpret_cast<const int *>(RB + ((int64_t)l * n + j) * kp);
    int acc = 0;
    for (int64_t h = 0; h < kp / 4; h++) acc = __dp4a(__ldg(a + h), __ldg(b + h), acc);
    const Oz2ModTab tb = c_mod[l];
    U[((int64_t)l * n + j) * mp + i] = (uint8_t)(l == 0 ? ((uint32_t)acc & 0xFFu) : mod_p_i32(acc, tb));
}

__global__ void k_mod_p(int l, const int32_t *__restrict__ in, uint8_t *__restrict__ out, int64_t count)
{
    int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= count) return;
    const Oz2ModTab tb = c_mod[l];
    out[t] = (uint8_t)(l == 0 ? ((uint32_t)in[t] & 0xFFu) : mod_p_i32(in[t], tb));
}

// planes [nplanes][rows][kp] INT8 -> 3-D map (k, row, plane), box (128, box_rows, 1), 128B swizzle, zero OOB fill
int make_plane_map(CUtensorMap *map, const int8_t *base, int64_t kp, int64_t rows, int nplanes, int box_rows)
{
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) return (int)cudaErrorNotSupported;
    cuuint64_t dims[3] = { (cuuint64_t)kp, (cuuint64_t)rows, (cuuint64_t)nplanes };
    cuuint64_t strides[2] = { (cuuint64_t)kp, (cuuint64_t)(rows * kp) };
    cuuint32_t box[3] = { (cuuint32_t)TILE_K, (cuuint32_t)box_rows, 1u };
    cuuint32_t estr[3] = { 1u, 1u, 1u };
    CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<int8_t *>(base), dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? 0 : (int)cudaErrorInvalidValue;
}

int num_sms()
{
    static int sms = 0;
    if (!sms) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    }
    return sms;
}

} // namespace

int oz2_gemm_upload_tables(const Oz2HostTables &t)
{
    OZ2_CUDA_TRY(cudaMemcpyToSymbol(c_mod, t.mod, sizeof(t.mod)));
    OZ2_CUDA_TRY(cudaFuncSetAttribute(k3_residue_gemm<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES));
    OZ2_CUDA_TRY(cudaFuncSetAttribute(k3_residue_gemm<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES));
    return 0;
}

int oz2_launch_gemm_tc(int nplanes, int mod_base, int64_t m, int64_t n, int64_t k, const int8_t *RA, const int8_t *RB,
                       int64_t kp, uint8_t *U, int64_t mp, int32_t *rowmax, int32_t *colmax, cudaStream_t st)
{
    (void)k;
    if (m <= 0 || n <= 0 || nplanes <= 0) return 0;
    CUtensorMap mapA, mapB;
    int rc = make_plane_map(&mapA, RA, kp, m, nplanes, TILE_M);
    if (rc) return rc;
    rc = make_plane_map(&mapB, RB, kp, n, nplanes, TILE_N);
    if (rc) return rc;
    const int64_t tiles = (int64_t)nplanes * ((m + TILE_M - 1) / TILE_M) * ((n + TILE_N - 1) / TILE_N);
    int grid = num_sms();
    if (tiles < grid) grid = (int)tiles;
    const int num_kb = (int)(kp / TILE_K);
    if (rowmax)
        k3_residue_gemm<true><<<grid, NUM_THREADS, SMEM_BYTES, st>>>(mapA, mapB, nplanes, mod_base, (int)m, (int)n, num_kb,
                                                                   nullptr, mp, rowmax, colmax);
    else
        k3_residue_gemm<false><<<grid, NUM_THREADS, SMEM_BYTES, st>>>(mapA, mapB, nplanes, mod_base, (int)m, (int)n, num_kb,
                                                                    U, mp, nullptr, nullptr);
    oz2_count_launches(1);
    OZ2_CUDA_TRY(cudaGetLastError());
    return 0;
}

int oz2_launch_gemm_check(int nplanes, int64_t m, int64_t n, int64_t k, const int8_t *RA, const int8_t *RB, int64_t kp,
                          uint8_t *U, int64_t mp, cudaStream_t st)
{
    (void)k;
    if (m <= 0 || n <= 0 || nplanes <= 0) return 0;
    dim3 grid((unsigned)((m + 31) / 32), (unsigned)((n + 7) / 8), (unsigned)nplanes);
    k3_check<<<grid, 256, 0, st>>>(nplanes, (int)m, (int)n, kp, RA, RB, U, mp);
    oz2_count_launches(1);
    OZ2_CUDA_TRY(cudaGetLastError());
    return 0;
}

int oz2_launch_mod_p(int l, const int32_t *in, uint8_t *out, int64_t count, cudaStream_t st)
{
    if (count <= 0) return 0;
    k_mod_p<<<(unsigned)((count + 255) / 256), 256, 0, st>>>(l, in, out, count);
    oz2_count_launches(1);
    OZ2_CUDA_TRY(cudaGetLastError());
    return 0;
}
