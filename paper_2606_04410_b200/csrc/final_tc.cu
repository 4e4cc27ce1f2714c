// A9, input-stationary: the last decoder stage (3x3 conv 64 -> 12, pixel-shuffle x2, clamp, crop, planar fp32) with the
// three COLUMNS of the 3x3 stencil folded into the N dimension of the GEMM and its three ROWS taken by the tensor core from
// shifted views of the same input tile.
//
//   R[p][dx*16 + n] = sum_dy sum_k X[p + 32 (dy - 1)][k] * W[dy][dx][n][k]   (tcgen05: M = 128 input pixels, N = 48, K = 3 x 64)
//   conv[n][y][x]   = b[n] + R[(y, x-1)][n] + R[(y, x)][16 + n] + R[(y, x+1)][32 + n]
//
// The output-stationary kernel (conv_halo_kernel<EPI_FINAL>) issues 36 MMAs of N = 16 per 128 pixels and sits at ~80 % of
// the shared-memory port ("A9 floor").  A first input-stationary version folded all nine taps into N
// (4 MMAs of N = 144 per 128 pixels), summed the column shifts with 72 warp shuffles per warp and the row shifts through a
// shared-memory exchange with a barrier between the 12 row warps; clock64 traces showed those warps, then (rows through
// shifted views, columns through the exchange) the shared-memory port the bound: MMA operand reads, TMA writes, exchange
// traffic and shuffles all cross it (about 320 KB per tile at 128 B per clock = the 2700-cycle tile period measured).
// Here a tile row is 32 consecutive pixels of 128 B, so "the pixel one row up / down" is the same buffer viewed from 4 KB
// earlier / later -- the row shift costs no data movement at all -- and what is left to the warps is the column shift
// between neighbouring lanes of ONE warp: 24 shuffles, no shared-memory exchange, no barrier, no coupling between warps.
//
// Tile = 16 rows x 32 columns of INPUT pixels (window origin one pixel up-left of the 14 x 30 output pixels it yields; 12 rows
// measured 173 us, 16 rows 159 us: one halo row in eight instead of one in six);
// one TMA box {64 ch, 32, 16} (zero-filled outside the image = the conv's zero padding) = four 128-row A operands.
// warp 0 = TMA producer, warp 1 = MMA issuer + TMEM allocator, warps 2..17 = one per tile row (group g = row / 4 reads
// accumulator g; warp % 4 = TMEM lane quadrant).  Accumulators are double-buffered over tiles (2 x 4 x 48 of 64 columns: all of
// TMEM), the weights of the current frame (18 KB) stay resident in shared memory.
#include <cuda.h>

#include "tc_ptx.cuh"
#include "ufnvc_internal.h"

namespace ufnvc {

namespace {

constexpr int kFG = 4;                                  // row groups (128-pixel MMA operands) per tile
constexpr int kFR = 4 * kFG, kFC = 32;                  // input rows / columns per tile
constexpr int kFOutR = kFR - 2, kFOutC = kFC - 2;       // output pixels per tile: 14 x 30
constexpr int kFN = 48;                                 // 3 stencil columns x 16 packed output columns
constexpr int kFAccStride = 64;                         // TMEM columns between accumulators (2 buffers x kFG row groups = 512 columns)
constexpr int kFThreads = (2 + kFR) * 32;
constexpr uint32_t kFABytes = kFR * kFC * 128;          // 65536: one input tile, 64 channels
constexpr uint32_t kFWBytes = 9 * 16 * 128;             // 18432: one frame's weights
constexpr uint32_t kFWdy = 3 * 16 * 128;                // 6144: the 48 rows [dx][n] of one stencil row
constexpr int kFAStages = 3;
// The weights sit BEFORE the input stages and 4 KB of padding after them: the views shifted by one tile row (-4 KB / +4 KB) of the
// first / last row group then read mapped shared memory (values that only reach the tile's halo rows, which produce no output).
constexpr uint32_t kFOffW = 0, kFOffA = kFWBytes, kFOffBar = kFOffA + kFAStages * kFABytes + 4096;
constexpr uint32_t kFSmem = kFOffBar + 256 + 1024;
static_assert(2 * kFG * kFAccStride <= 512 && kFSmem <= 227 * 1024, "accumulators fit TMEM, the stages fit shared memory");

struct FDiv {                                            // division by a runtime constant (tile index -> coordinates)
    uint32_t d, mul, shr;
    __device__ __forceinline__ uint32_t div(uint32_t n) const { return (__umulhi(n, mul) + n) >> shr; }
};
FDiv make_fdiv(uint32_t d)
{
    FDiv f;
    f.d = d;
    uint32_t l = 0;
    while ((1ull << l) < d) ++l;
    f.mul = uint32_t(((1ull << 32) * ((1ull << l) - d)) / d + 1);
    f.shr = l;
    return f;
}

struct FinalParams {
    int n_img, H, W;             // input images (NHWC bf16, 64 channels)
    int tiles_y, tiles_x, total_tiles;
    FDiv fd_tx, fd_ty, fd_groups;
    int groups;                  // weight sets (frame index = img % groups)
    const float *bias;           // [groups][16]
    float *out;                  // [n_img][3][out_h][out_w]
    int out_h, out_w;
};

enum : uint32_t {
    F_AFULL = 0, F_AEMPTY = F_AFULL + kFAStages, F_WFULL = F_AEMPTY + kFAStages, F_WFREE = F_WFULL + 1, F_DFULL = F_WFREE + 1,
    F_DEMPTY = F_DFULL + 2 * kFG, F_TMEM = F_DEMPTY + 2 * kFG
};

}  // namespace

namespace {

struct FTile { int img, y0, x0, grp; };     // (y0, x0) = input-window origin = output-tile origin - 1
__device__ __forceinline__ FTile f_tile(const FinalParams &p, int tile)
{
    FTile t;
    const uint32_t r = p.fd_tx.div(uint32_t(tile)), tx = uint32_t(tile) - r * p.fd_tx.d;
    const uint32_t img = p.fd_ty.div(r), ty = r - img * p.fd_ty.d;
    t.img = int(img);
    t.y0 = int(ty) * kFOutR - 1;
    t.x0 = int(tx) * kFOutC - 1;
    t.grp = p.groups == 1 ? 0 : int(img - p.fd_groups.div(img) * p.fd_groups.d);
    return t;
}

__global__ void __launch_bounds__(kFThreads, 1)
final_is_kernel(const __grid_constant__ CUtensorMap tm_in, const __grid_constant__ CUtensorMap tm_w, const FinalParams p)
{
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    auto bar = [&](uint32_t slot) { return base + kFOffBar + 8u * slot; };
    volatile uint32_t *tmem_slot_ptr = reinterpret_cast<volatile uint32_t *>(smem_raw + (bar(F_TMEM) - smem_u32(smem_raw)));
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_in) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_w) : "memory");
        for (int s = 0; s < kFAStages; ++s) { mbar_init(bar(F_AFULL + s), 1); mbar_init(bar(F_AEMPTY + s), 1); }
        mbar_init(bar(F_WFULL), 1); mbar_init(bar(F_WFREE), 1);
        for (int a = 0; a < 2 * kFG; ++a) { mbar_init(bar(F_DFULL + a), 1); mbar_init(bar(F_DEMPTY + a), 4); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(bar(F_TMEM)), "r"(512u) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;
    pdl_grid_sync();                                                 // the predecessor kernel's output is complete and visible from here on

    if (warp == 0) {
        // ===================== TMA producer =====================
        if (elect_one()) {
            int sa = 0; uint32_t pa = 0, pfree = 0;
            int prev_grp = -1;
            for (int tile = blockIdx.x; tile < p.total_tiles; tile += gridDim.x) {
                const FTile t = f_tile(p, tile);
                if (t.grp != prev_grp) {
                    // this frame's weights, resident: [dy][dx][16 n][64 k] -- the 48 rows (dx, n) of one stencil row dy are one B operand
                    if (prev_grp >= 0) { mbar_wait(bar(F_WFREE), pfree); pfree ^= 1; }
                    mbar_expect_tx(bar(F_WFULL), kFWBytes);
                    tma_load_3d(base + kFOffW, &tm_w, bar(F_WFULL), 0, 0, t.grp);
                    prev_grp = t.grp;
                }
                mbar_wait(bar(F_AEMPTY + sa), pa ^ 1);
                mbar_expect_tx(bar(F_AFULL + sa), kFABytes);
                tma_load_4d(base + kFOffA + uint32_t(sa) * kFABytes, &tm_in, bar(F_AFULL + sa), 0, t.x0, t.y0, t.img);
                if (++sa == kFAStages) { sa = 0; pa ^= 1; }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer: per tile 3 row groups x (3 row shifts x 4 k-steps) of N = 48 =====================
        if (elect_one()) {
            const uint32_t idesc = umma_idesc_bf16(128, kFN);
            const uint32_t hi = uint32_t(1024 >> 4) | (1u << 14) | (2u << 29);
            const uint32_t a_lo0 = (((base + kFOffA) & 0x3FFFFu) >> 4) | (1u << 16);
            const uint32_t w_lo = (((base + kFOffW) & 0x3FFFFu) >> 4) | (1u << 16);
            int sa = 0; uint32_t pa = 0, pw = 0;
            int prev_grp = -1, it = 0;
            for (int tile = blockIdx.x; tile < p.total_tiles; tile += gridDim.x, ++it) {
                const FTile t = f_tile(p, tile);
                if (t.grp != prev_grp) { mbar_wait(bar(F_WFULL), pw); pw ^= 1; prev_grp = t.grp; }
                mbar_wait(bar(F_AFULL + sa), pa);
                tc_fence_after();
                const uint32_t a_lo = a_lo0 + uint32_t(sa) * (kFABytes >> 4);
                const int buf = it & 1;
#pragma unroll
                for (int g = 0; g < kFG; ++g) {
                    mbar_wait(bar(F_DEMPTY + kFG * buf + g), ((it >> 1) & 1) ^ 1);   // the row warps of group g have drained this accumulator
                    tc_fence_after();
#pragma unroll
                    for (int dy = 0; dy < 3; ++dy)
#pragma unroll
                        for (int k = 0; k < 4; ++k)                               // view shifted by dy - 1 tile rows = (dy - 1) * 4096 B = 256 units
                            umma_bf16_lh(tmem_base + uint32_t((kFG * buf + g) * kFAccStride),
                                         a_lo + uint32_t(g) * (16384 >> 4) + uint32_t(256 * dy) - 256u + 2 * k, hi,
                                         w_lo + uint32_t(dy) * (kFWdy >> 4) + 2 * k, hi, idesc, uint32_t(dy | k));
                    umma_commit(bar(F_DFULL + kFG * buf + g));
                }
                umma_commit(bar(F_AEMPTY + sa));
                if (++sa == kFAStages) { sa = 0; pa ^= 1; }
                const int next = tile + gridDim.x;
                if (next < p.total_tiles && f_tile(p, next).grp != prev_grp) umma_commit(bar(F_WFREE));
            }
        }
    } else {
        // ===================== row warps 2..13: one tile row each =====================
        const int q = warp & 3, g = (warp - 2) >> 2;                       // TMEM lane quadrant (a hardware rule), row group
        const int r = 4 * g + q, cx = lane;
        const uint32_t t_row = tmem_base + (uint32_t(q * 32) << 16);
        auto ld16 = [](uint32_t taddr, uint32_t (&v)[16]) {
            asm volatile(
                "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
                "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
                  "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                : "r"(taddr));
        };
        int it = 0, bias_grp = -1;
        float bs[12];
        for (int tile = blockIdx.x; tile < p.total_tiles; tile += gridDim.x, ++it) {
            const FTile t = f_tile(p, tile);
            if (t.grp != bias_grp) {                                       // (L1 is a few KB here: keep the bias out of the tile loop)
#pragma unroll
                for (int n = 0; n < 12; ++n) bs[n] = __ldg(p.bias + t.grp * 16 + n);
                bias_grp = t.grp;
            }
            const int buf = it & 1;
            mbar_wait(bar(F_DFULL + kFG * buf + g), (it >> 1) & 1);
            tc_fence_after();
            // R_dx of this pixel: columns [16 dx, 16 dx + 12) of the accumulator.  The output pixel (y, x) takes R_0 from the pixel to
            // its left and R_2 from the pixel to its right: the neighbouring lanes of this warp.
            uint32_t r0[16], r1[16], r2[16];
            const uint32_t t_acc = t_row + uint32_t((kFG * buf + g) * kFAccStride);
            ld16(t_acc, r0);
            ld16(t_acc + 16, r1);
            ld16(t_acc + 32, r2);
            tmem_ld_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(F_DEMPTY + kFG * buf + g));        // the accumulator may be overwritten (by tile it + 2)
            float o[12];
#pragma unroll
            for (int n = 0; n < 12; ++n)
                o[n] = bs[n] + __shfl_up_sync(0xFFFFFFFFu, __uint_as_float(r0[n]), 1) + __uint_as_float(r1[n]) +
                       __shfl_down_sync(0xFFFFFFFFu, __uint_as_float(r2[n]), 1);
            const int y = t.y0 + r, x = t.x0 + cx;
            if (r >= 1 && r <= kFOutR && cx >= 1 && cx <= kFOutC && y < p.H && x < p.W) {
                // packed column n = (2i + j) * 3 + c -> out[img][c][2y + i][2x + j] (R14), clamp (O9), crop
                float *ob = p.out + (long long)t.img * 3 * p.out_h * p.out_w;
                const int ox = 2 * x;
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    const int oy = 2 * y + i;
                    if (oy >= p.out_h) continue;
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const float a = fminf(fmaxf(o[(2 * i) * 3 + c], 0.0f), 1.0f), b = fminf(fmaxf(o[(2 * i + 1) * 3 + c], 0.0f), 1.0f);
                        float *dst = ob + ((long long)c * p.out_h + oy) * p.out_w + ox;
                        if (ox + 1 < p.out_w) *reinterpret_cast<float2 *>(dst) = make_float2(a, b);
                        else if (ox < p.out_w) *dst = a;
                    }
                }
            }
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512u) : "memory");
    }
}

}  // namespace

// ---------------------------------------------------------------- host side ----------------------------------
bool final_is_eligible(const ConvLayer &L, int out_w)
{
    return L.c_in == 64 && L.n == 12 && L.n_pad == 16 && L.taps == 9 && (out_w % 2) == 0;
}

bool final_make_maps(FinalMaps &m, const ConvLayer &L, const bf16 *in_base, int n_img, int H, int W, int out_w, std::string &err)
{
    m.ok = false;
    if (!final_is_eligible(L, out_w)) return true;
    if (!tc_make_act_tmap(&m.tm_in, in_base, n_img, H, W, 64, kFR, kFC, err)) return false;
    // weights [group][tap][16][64] bf16 are [group][144][64]: one box = one frame's whole weight set
    if (!tc_encode_3d(&m.tm_w, L.w, 64, 144, (unsigned long long)L.groups, 64, 144, 1, err)) return false;
    m.ok = true;
    return true;
}

cudaError_t configure_final_kernels()
{
    return cudaFuncSetAttribute(final_is_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, int(kFSmem));
}

cudaError_t launch_final_is(const FinalMaps &m, const ConvLayer &L, int n_img, int H, int W, float *out, int out_h, int out_w,
                            int num_sms, LaunchStream st)
{
    FinalParams p{};
    p.n_img = n_img; p.H = H; p.W = W;
    p.tiles_y = (H + kFOutR - 1) / kFOutR;
    p.tiles_x = (W + kFOutC - 1) / kFOutC;
    p.total_tiles = n_img * p.tiles_y * p.tiles_x;
    p.fd_tx = make_fdiv(uint32_t(p.tiles_x)); p.fd_ty = make_fdiv(uint32_t(p.tiles_y)); p.fd_groups = make_fdiv(uint32_t(L.groups));
    p.groups = L.groups;
    p.bias = L.bias;
    p.out = out; p.out_h = out_h; p.out_w = out_w;
    const int grid = p.total_tiles < num_sms ? p.total_tiles : num_sms;
    return launch_pdl(final_is_kernel, grid, kFThreads, kFSmem, st, 1, m.tm_in, m.tm_w, p);
}

}  // namespace ufnvc
