// tcgen05 implicit-GEMM convolution for sm_100a (north_star: "implicit-GEMM 3x3 and 1x1
// convolutions on tcgen05/TMEM tensor cores fed by TMA, with bias, activation and pixel-shuffle upsampling fused into
// the epilogue ... the frame-specific decoders as one grouped-weight launch over the T frame indices").
//
//   D[128 pixels][BN out-channels] (fp32, TMEM) += A[128 pixels][64 ch] (bf16, smem) * B[BN][64 ch]^T (bf16, smem)
//   summed over 9 taps (or 1) x (C_in / 64) channel slabs.
//
//   * A: one TMA box {64 ch, TW, TH, 1 img} of the NHWC activation per (tap, slab), at SIGNED coordinates
//     (x0 + dx - 1, y0 + dy - 1): out-of-bounds rows/columns are zero-filled by the TMA unit, which is the conv's
//     zero padding -- no halo code, no im2col buffer.  128-byte swizzle; box row r lands at r * 128 B, which is
//     exactly the K-major SWIZZLE_128B operand layout tcgen05.mma reads (8-row groups 1024 B apart).
//   * B: TMA box {64 ch, BN rows, 1} of w[group][tap][n][c_in]; group = image index mod T selects the frame-specific
//     weight set, so one launch covers all T decoders.
//   * warp 0 = TMA producer, warp 1 = MMA issuer (one elected thread) + TMEM allocator, warps 2..5 = epilogue
//     (tcgen05.ld -> bias -> GELU -> bf16 -> pixel-shuffle / NHWC / final planar store).  4-stage smem ring,
//     2 TMEM accumulator stages so the epilogue of tile i overlaps the MMAs of tile i+1.  Persistent: grid = #SMs.
#include <cuda.h>

#include "epilogue.cuh"
#include "ufnvc_internal.h"

namespace ufnvc {

namespace {

constexpr int kStages = 4;
constexpr int kTileM = 128;
constexpr int kSlabK = 64;                       // bf16 channels per smem row = 128 bytes = one swizzle span
constexpr int kABytes = kTileM * kSlabK * 2;     // 16 KB
constexpr int kThreads = 192;
constexpr uint32_t kSpinLimit = 1u << 28;

struct TcParams {
    int n_img_m, Hm, Wm;          // activation as the TMA map sees it (flattened for 1x1 convs)
    int tiles_y, tiles_x, TH, TW;
    int H, W;                     // real image dims: global pixel -> (img, y, x) for the epilogue
    int taps, slabs;              // k-blocks per tile = taps * slabs
    int n_tiles, BN, n_real, n_pad;
    int groups;
    int total_tiles;
    const float *bias;            // [groups][n_pad]
    EpiParams E;
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok = 0, spins = 0;
    while (true) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok)
            : "r"(bar), "r"(parity)
            : "memory");
        if (ok) return;
        if (++spins > kSpinLimit) __trap();      // a protocol bug must fail loudly, never hang the GPU
    }
}

__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap *tm, uint32_t bar, int c0, int c1, int c2, int c3)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
        ::"r"(dst), "l"(tm), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
        : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap *tm, uint32_t bar, int c0, int c1, int c2)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(dst), "l"(tm), "r"(bar), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
}

// K-major, SWIZZLE_128B shared-memory matrix descriptor (PTX ISA "tcgen05 matrix descriptor"):
//   [0,14) start address >> 4, [16,30) leading byte offset >> 4 (unused for swizzled K-major; 1),
//   [32,46) stride byte offset >> 4 (8 rows x 128 B = 1024 -> 64), [46,48) version = 1, [61,64) layout = 2 (128B).
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t saddr)
{
    return uint64_t((saddr & 0x3FFFFu) >> 4) | (uint64_t(1) << 16) | (uint64_t(1024 >> 4) << 32) | (uint64_t(1) << 46) |
           (uint64_t(2) << 61);
}

// kind::f16 instruction descriptor: D = f32 (bits [4,6) = 1), A = B = bf16 ([7,10) = [10,13) = 1), both K-major,
// N >> 3 at [17,23), M >> 4 at [24,29).
__device__ __forceinline__ uint32_t umma_idesc_bf16(int M, int N)
{
    return (1u << 4) | (1u << 7) | (1u << 10) | (uint32_t(N >> 3) << 17) | (uint32_t(M >> 4) << 24);
}

__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }

__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]),
          "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]),
          "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

}  // namespace

namespace {

// tile index -> (image in map space, tile origin, n tile); n fastest so CTAs running side by side share the A tile in L2
struct TileCoord { int img, y0, x0, nt; };
__device__ __forceinline__ TileCoord tile_coord(const TcParams &p, int tile)
{
    TileCoord c;
    c.nt = tile % p.n_tiles;
    int r = tile / p.n_tiles;
    const int tx = r % p.tiles_x; r /= p.tiles_x;
    const int ty = r % p.tiles_y;
    c.img = r / p.tiles_y;
    c.y0 = ty * p.TH;
    c.x0 = tx * p.TW;
    return c;
}

template <int MODE>
__global__ void __launch_bounds__(kThreads, 1)
conv_tc_kernel(const __grid_constant__ CUtensorMap tmap_a, const __grid_constant__ CUtensorMap tmap_b, const TcParams p)
{
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    // carve: [stages][A 16 KB | B BN*128] (1024-aligned), then barriers
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t b_bytes = uint32_t(p.BN) * 128u;
    const uint32_t stage_bytes = kABytes + b_bytes;                 // multiple of 1024 (BN multiple of 16 -> 2 KB)
    const uint32_t bar_base = smem_base + kStages * stage_bytes;
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (kStages + s); };
    auto tfull_bar = [&](int a) { return bar_base + 8u * (2 * kStages + a); };
    auto tempty_bar = [&](int a) { return bar_base + 8u * (2 * kStages + 2 + a); };
    const uint32_t tmem_slot = bar_base + 8u * (2 * kStages + 4);
    volatile uint32_t *tmem_slot_ptr = reinterpret_cast<volatile uint32_t *>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int kblocks = p.taps * p.slabs;
    uint32_t tmem_cols = 32;
    while (tmem_cols < uint32_t(2 * p.BN)) tmem_cols <<= 1;

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmap_a) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmap_b) : "memory");
        for (int s = 0; s < kStages; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
        for (int a = 0; a < 2; ++a) { mbar_init(tfull_bar(a), 1); mbar_init(tempty_bar(a), 4); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "r"(tmem_cols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    if (warp == 0) {
        // ===================== TMA producer =====================
        if (lane == 0) {
            int stage = 0; uint32_t phase = 0;
            for (int tile = blockIdx.x; tile < p.total_tiles; tile += gridDim.x) {
                const TileCoord tc = tile_coord(p, tile);
                const int grp = p.groups == 1 ? 0 : tc.img % p.groups;
                for (int kb = 0; kb < kblocks; ++kb) {
                    const int tap = kb / p.slabs, slab = kb - tap * p.slabs;
                    const int dy = p.taps == 9 ? tap / 3 - 1 : 0, dx = p.taps == 9 ? tap % 3 - 1 : 0;
                    mbar_wait(empty_bar(stage), phase ^ 1);
                    const uint32_t a_dst = smem_base + stage * stage_bytes, b_dst = a_dst + kABytes;
                    mbar_expect_tx(full_bar(stage), stage_bytes);
                    tma_load_4d(a_dst, &tmap_a, full_bar(stage), slab * kSlabK, tc.x0 + dx, tc.y0 + dy, tc.img);
                    tma_load_3d(b_dst, &tmap_b, full_bar(stage), slab * kSlabK, tc.nt * p.BN, grp * p.taps + tap);
                    if (++stage == kStages) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer =====================
        if (lane == 0) {
            const uint32_t idesc = umma_idesc_bf16(kTileM, p.BN);
            int stage = 0; uint32_t phase = 0;
            int it = 0;
            for (int tile = blockIdx.x; tile < p.total_tiles; tile += gridDim.x, ++it) {
                const int acc = it & 1;
                const uint32_t acc_phase = (it >> 1) & 1;
                mbar_wait(tempty_bar(acc), acc_phase ^ 1);            // epilogue has drained this accumulator
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + uint32_t(acc * p.BN);
                for (int kb = 0; kb < kblocks; ++kb) {
                    mbar_wait(full_bar(stage), phase);
                    tc_fence_after();
                    const uint32_t a_src = smem_base + stage * stage_bytes, b_src = a_src + kABytes;
                    const uint64_t da = umma_desc_sw128(a_src), db = umma_desc_sw128(b_src);
#pragma unroll
                    for (int k = 0; k < kSlabK / 16; ++k)           // 16 bf16 = 32 bytes = +2 in descriptor units
                        umma_bf16(d_tmem, da + uint64_t(2 * k), db + uint64_t(2 * k), idesc, (kb | k) != 0);
                    umma_commit(empty_bar(stage));                   // frees the smem stage when these MMAs retire
                    if (kb == kblocks - 1) umma_commit(tfull_bar(acc));
                    if (++stage == kStages) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else {
        // ===================== epilogue: 4 warps, warp w owns TMEM lanes 32*(w%4) .. +31 =====================
        const int quad = warp & 3;
        const int m = quad * 32 + lane;                               // accumulator row = pixel inside the tile
        const int P = p.H * p.W;
        int it = 0;
        for (int tile = blockIdx.x; tile < p.total_tiles; tile += gridDim.x, ++it) {
            const TileCoord tc = tile_coord(p, tile);
            const int acc = it & 1;
            const uint32_t acc_phase = (it >> 1) & 1;
            const int ym = tc.y0 + m / p.TW, xm = tc.x0 + m % p.TW;
            const bool inb = ym < p.Hm && xm < p.Wm;
            // map-space pixel -> real (img, y, x)
            const long long gp = ((long long)tc.img * p.Hm + ym) * p.Wm + xm;
            const int img = int(gp / P);
            const int rem = int(gp - (long long)img * P);
            const int y = rem / p.W, x = rem - y * p.W;
            const int grp = p.groups == 1 ? 0 : img % p.groups;
            const float *bias = p.bias + (long long)grp * p.n_pad + tc.nt * p.BN;
            mbar_wait(tfull_bar(acc), acc_phase);
            tc_fence_after();
            const uint32_t t_row = tmem_base + (uint32_t(quad * 32) << 16) + uint32_t(acc * p.BN);
            if (MODE == EPI_FINAL) {
                uint32_t v[16];
                tmem_ld16(t_row, v);
                if (inb) {
#pragma unroll
                    for (int j = 0; j < 16; ++j) {
                        const int n = tc.nt * p.BN + j;
                        if (n < p.n_real) epi_store_final(p.E, img, y, x, n, __uint_as_float(v[j]) + __ldg(bias + j));
                    }
                }
            } else {
                for (int c0 = 0; c0 < p.BN; c0 += 32) {
                    uint32_t v[32];
                    tmem_ld32(t_row + uint32_t(c0), v);
                    if (!inb) continue;
                    const int n = tc.nt * p.BN + c0;                  // 32 consecutive packed columns, one store run
                    const long long o = epi_offset(p.E, img, y, x, p.H, p.W, n);
                    bf16 *dst = reinterpret_cast<bf16 *>(p.E.out) + o;
                    float f[32];
#pragma unroll
                    for (int j = 0; j < 32; j += 4) {
                        const float4 b4 = __ldg(reinterpret_cast<const float4 *>(bias + c0 + j));
                        f[j] = __uint_as_float(v[j]) + b4.x; f[j + 1] = __uint_as_float(v[j + 1]) + b4.y;
                        f[j + 2] = __uint_as_float(v[j + 2]) + b4.z; f[j + 3] = __uint_as_float(v[j + 3]) + b4.w;
                    }
                    if (p.E.act == ACT_GELU) {
#pragma unroll
                        for (int j = 0; j < 32; ++j) f[j] = gelu_erf(f[j]);
                    }
                    if (MODE == EPI_NHWC && p.E.residual) {
                        const uint4 *rs = reinterpret_cast<const uint4 *>(p.E.residual + o);
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            const uint4 r4 = rs[q];
                            const bf16 *re = reinterpret_cast<const bf16 *>(&r4);
#pragma unroll
                            for (int e = 0; e < 8; ++e) f[q * 8 + e] += __bfloat162float(re[e]);
                        }
                    }
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        uint4 o4;
                        __nv_bfloat162 *oe = reinterpret_cast<__nv_bfloat162 *>(&o4);
#pragma unroll
                        for (int e = 0; e < 4; ++e) oe[e] = __floats2bfloat162_rn(f[q * 8 + 2 * e], f[q * 8 + 2 * e + 1]);
                        reinterpret_cast<uint4 *>(dst)[q] = o4;
                    }
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tempty_bar(acc));
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(tmem_cols) : "memory");
    }
}

}  // namespace

// ---------------------------------------------------------------- host side ----------------------------------
namespace {
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_fn()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}
bool encode(CUtensorMap *tm, const void *base, int rank, const cuuint64_t *dims, const cuuint64_t *strides_bytes, const cuuint32_t *box,
            std::string &err)
{
    EncodeTiledFn fn = encode_fn();
    if (!fn) { err = "cuTensorMapEncodeTiled entry point not found"; return false; }
    cuuint32_t ones[5] = {1, 1, 1, 1, 1};
    CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, rank, const_cast<void *>(base), dims, strides_bytes, box, ones,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { err = "cuTensorMapEncodeTiled failed: " + std::to_string(int(r)); return false; }
    return true;
}
int pick_block_n(int n_pad)
{
    for (int bn = 256; bn >= 16; bn -= 16)
        if (n_pad % bn == 0) return bn;
    return 0;
}
}  // namespace

bool tc_make_weight_tmap(ConvLayer &L, std::string &err)
{
    L.use_tc = false;
    if (L.c_in % kSlabK || L.n_pad % 16) return true;                  // not eligible: stays on the CUDA-core kernel
    L.block_n = pick_block_n(L.n_pad);
    if (L.block_n != 16 && L.block_n % 32) return true;                // epilogue works on 32-column runs
    cuuint64_t dims[3] = {cuuint64_t(L.c_in), cuuint64_t(L.n_pad), cuuint64_t(L.groups) * L.taps};
    cuuint64_t strides[2] = {cuuint64_t(L.c_in) * 2, cuuint64_t(L.c_in) * 2 * L.n_pad};
    cuuint32_t box[3] = {cuuint32_t(kSlabK), cuuint32_t(L.block_n), 1};
    if (!encode(&L.tmap_w, L.w, 3, dims, strides, box, err)) return false;
    L.use_tc = true;
    return true;
}

bool tc_make_act_tmap(CUtensorMap *tm, const bf16 *base, int n_img, int H, int W, int C, int tile_h, int tile_w, std::string &err)
{
    cuuint64_t dims[4] = {cuuint64_t(C), cuuint64_t(W), cuuint64_t(H), cuuint64_t(n_img)};
    cuuint64_t strides[3] = {cuuint64_t(C) * 2, cuuint64_t(C) * 2 * W, cuuint64_t(C) * 2 * W * H};
    cuuint32_t box[4] = {cuuint32_t(kSlabK), cuuint32_t(tile_w), cuuint32_t(tile_h), 1};
    return encode(tm, base, 4, dims, strides, box, err);
}

cudaError_t launch_conv_tc(const ConvLayer &L, const ConvProblem &P, const CUtensorMap &tmap_in, int tile_h, int tile_w, bool flat,
                           const EpiParams &E, int num_sms, cudaStream_t st)
{
    TcParams p{};
    p.H = P.H; p.W = P.W;
    if (flat) {                                   // 1x1 conv: pixels of all images as rows of a [total/128][128] "image"
        const long long total = (long long)P.n_img * P.H * P.W;
        if (L.taps != 1 || total % kTileM) return cudaErrorInvalidValue;
        p.n_img_m = 1; p.Hm = int(total / kTileM); p.Wm = kTileM;
    } else {
        p.n_img_m = P.n_img; p.Hm = P.H; p.Wm = P.W;
    }
    p.TH = tile_h; p.TW = tile_w;
    p.tiles_y = (p.Hm + tile_h - 1) / tile_h;
    p.tiles_x = (p.Wm + tile_w - 1) / tile_w;
    p.taps = L.taps; p.slabs = L.c_in / kSlabK;
    p.BN = L.block_n; p.n_tiles = L.n_pad / L.block_n; p.n_real = L.n; p.n_pad = L.n_pad;
    p.groups = L.groups;
    p.total_tiles = p.n_img_m * p.tiles_y * p.tiles_x * p.n_tiles;
    p.bias = L.bias;
    p.E = E;
    const size_t smem = size_t(kStages) * (kABytes + size_t(L.block_n) * 128) + 1024 + 256;
    const int grid = p.total_tiles < num_sms ? p.total_tiles : num_sms;
    auto launch = [&](auto kern) -> cudaError_t {
        static thread_local const void *configured[8] = {};
        bool done = false;
        for (const void *c : configured) done |= (c == (const void *)kern);
        if (!done) {
            cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
            if (e != cudaSuccess) return e;
            for (auto &c : configured) if (!c) { c = (const void *)kern; break; }
        }
        kern<<<grid, kThreads, smem, st>>>(tmap_in, L.tmap_w, p);
        return cudaGetLastError();
    };
    switch (E.mode) {
        case EPI_NHWC: return launch(conv_tc_kernel<EPI_NHWC>);
        case EPI_PS2: return launch(conv_tc_kernel<EPI_PS2>);
        default: return launch(conv_tc_kernel<EPI_FINAL>);
    }
}

}  // namespace ufnvc
