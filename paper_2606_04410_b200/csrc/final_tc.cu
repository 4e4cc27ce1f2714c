// A9, input-stationary: the last decoder stage (3x3 conv 64 -> 12, pixel-shuffle x2, clamp, crop, planar fp32) with the
// nine taps folded into the N dimension of ONE GEMM per input pixel.
//
//   P[p][tap*16 + n] = sum_k X[p][k] * W[tap][n][k]           (tcgen05: M = 128 input pixels, N = 144, K = 64)
//   conv[n][y][x]    = b[n] + sum_{dy,dx} P[(y+dy-1, x+dx-1)][(3 dy + dx)*16 + n]
//
// The output-stationary kernel (conv_halo_kernel<EPI_FINAL>) issues 36 MMAs of N = 16 per 128 pixels and every one of
// them fetches a 4 KB A operand: it sits at ~80 % of the shared-memory port ("A9 floor").  Here
// 128 input pixels cost 4 MMAs (9x fewer operand bytes); the price is a shifted sum of the nine partial planes, which
// lives in different TMEM lanes (= pixels): dx by warp shuffles (a warp is one row of 32 pixels), dy through a small
// shared-memory exchange between the 12 row-warps of a tile.
//
// Tile = 12 rows x 32 columns of INPUT pixels (window origin one pixel up-left of the 10 x 30 output pixels it yields);
// one TMA box {64 ch, 32, 12} (zero-filled outside the image = the conv's zero padding) = three 128-row A operands.
// warp 0 = TMA producer, warp 1 = MMA issuer + TMEM allocator, warps 2..13 = one per tile row (group g = row / 4 reads
// accumulator g; warp % 4 = TMEM lane quadrant).  Weights of the current frame (18 KB) stay resident in shared memory.
#include <cuda.h>

#include "tc_ptx.cuh"
#include "ufnvc_internal.h"

namespace ufnvc {

namespace {

constexpr int kFR = 12, kFC = 32;                       // input rows / columns per tile
constexpr int kFOutR = kFR - 2, kFOutC = kFC - 2;       // output pixels per tile: 10 x 30
constexpr int kFN = 144;                                // 9 taps x 16 packed output columns
constexpr int kFThreads = 14 * 32;
constexpr uint32_t kFABytes = kFR * kFC * 128;          // 49152: one input tile, 64 channels
constexpr uint32_t kFWBytes = kFN * 128;                // 18432: one frame's weights
constexpr int kFAStages = 2;
constexpr uint32_t kFXQ = kFR * kFC * 16 * 6;           // exchange buffer: 6 float4 planes x 384 pixels = 36864 B
constexpr uint32_t kFOffW = kFAStages * kFABytes, kFOffXQ = kFOffW + 2 * 18432, kFOffBar = kFOffXQ + 2 * kFXQ;
constexpr uint32_t kFSmem = kFOffBar + 256 + 1024;

struct FinalParams {
    int n_img, H, W;             // input images (NHWC bf16, 64 channels)
    int tiles_y, tiles_x, total_tiles;
    int groups;                  // weight sets (frame index = img % groups)
    const float *bias;           // [groups][16]
    float *out;                  // [n_img][3][out_h][out_w]
    int out_h, out_w;
};

enum : uint32_t { F_AFULL = 0, F_AEMPTY = 2, F_WFULL = 4, F_WFREE = 5, F_DFULL = 6, F_DEMPTY = 9, F_TMEM = 12 };

}  // namespace

namespace {

struct FTile { int img, y0, x0, grp; };     // (y0, x0) = input-window origin = output-tile origin - 1
__device__ __forceinline__ FTile f_tile(const FinalParams &p, int tile)
{
    FTile t;
    const int tx = tile % p.tiles_x;
    const int r = tile / p.tiles_x;
    const int ty = r % p.tiles_y;
    t.img = r / p.tiles_y;
    t.y0 = ty * kFOutR - 1;
    t.x0 = tx * kFOutC - 1;
    t.grp = p.groups == 1 ? 0 : t.img % p.groups;
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
        for (int g = 0; g < 3; ++g) { mbar_init(bar(F_DFULL + g), 1); mbar_init(bar(F_DEMPTY + g), 4); }
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
                if (t.grp != prev_grp) {                                  // this frame's weights: [144 rows][64 k], resident
                    if (prev_grp >= 0) { mbar_wait(bar(F_WFREE), pfree); pfree ^= 1; }
                    mbar_expect_tx(bar(F_WFULL), kFWBytes);
                    tma_load_3d(base + kFOffW, &tm_w, bar(F_WFULL), 0, 0, t.grp);
                    prev_grp = t.grp;
                }
                mbar_wait(bar(F_AEMPTY + sa), pa ^ 1);
                mbar_expect_tx(bar(F_AFULL + sa), kFABytes);
                tma_load_4d(base + uint32_t(sa) * kFABytes, &tm_in, bar(F_AFULL + sa), 0, t.x0, t.y0, t.img);
                if (++sa == kFAStages) { sa = 0; pa ^= 1; }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer: 3 accumulators (row groups) x 4 k-steps of N = 144 =====================
        if (elect_one()) {
            const uint32_t idesc = umma_idesc_bf16(128, kFN);
            const uint32_t hi = uint32_t(1024 >> 4) | (1u << 14) | (2u << 29);
            const uint32_t a_lo0 = ((base & 0x3FFFFu) >> 4) | (1u << 16);
            const uint32_t w_lo = (((base + kFOffW) & 0x3FFFFu) >> 4) | (1u << 16);
            int sa = 0; uint32_t pa = 0, pw = 0;
            int prev_grp = -1, it = 0;
            for (int tile = blockIdx.x; tile < p.total_tiles; tile += gridDim.x, ++it) {
                const FTile t = f_tile(p, tile);
                if (t.grp != prev_grp) { mbar_wait(bar(F_WFULL), pw); pw ^= 1; prev_grp = t.grp; }
                mbar_wait(bar(F_AFULL + sa), pa);
                tc_fence_after();
                const uint32_t a_lo = a_lo0 + uint32_t(sa) * (kFABytes >> 4);
#pragma unroll
                for (int g = 0; g < 3; ++g) {
                    mbar_wait(bar(F_DEMPTY + g), (it & 1) ^ 1);           // the row warps of group g have drained accumulator g
                    tc_fence_after();
#pragma unroll
                    for (int k = 0; k < 4; ++k)
                        umma_bf16_lh(tmem_base + uint32_t(g * kFN), a_lo + uint32_t(g) * (16384 >> 4) + 2 * k, hi, w_lo + 2 * k, hi, idesc,
                                     uint32_t(k));
                    umma_commit(bar(F_DFULL + g));
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
        const uint32_t t_addr = tmem_base + (uint32_t(q * 32) << 16) + uint32_t(g * kFN);
        const uint32_t pix = uint32_t(r * kFC + cx);
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
            mbar_wait(bar(F_DFULL + g), it & 1);
            tc_fence_after();
            // Q_dy[n] = sum_dx P[(r, cx + dx - 1)][(dy, dx)][n]: the two side terms come from the neighbouring lanes.  Q_0 and
            // Q_2 are needed by rows r+1 / r-1, i.e. by other warps: they go straight to shared memory (6 float4 planes x 384
            // pixels, double-buffered over tiles); only Q_1 stays in registers.
            const uint32_t xq = base + kFOffXQ + uint32_t(it & 1) * kFXQ;
            float Q1[12];
#pragma unroll
            for (int dy = 0; dy < 3; ++dy) {
                uint32_t v0[16], v1[16], v2[16];
                ld16(t_addr + uint32_t((dy * 3 + 0) * 16), v0);
                ld16(t_addr + uint32_t((dy * 3 + 1) * 16), v1);
                ld16(t_addr + uint32_t((dy * 3 + 2) * 16), v2);
                tmem_ld_wait();
                float Qd[12];
#pragma unroll
                for (int n = 0; n < 12; ++n)
                    Qd[n] = __shfl_up_sync(0xFFFFFFFFu, __uint_as_float(v0[n]), 1) + __uint_as_float(v1[n]) +
                            __shfl_down_sync(0xFFFFFFFFu, __uint_as_float(v2[n]), 1);
                if (dy == 1) {
#pragma unroll
                    for (int n = 0; n < 12; ++n) Q1[n] = Qd[n];
                } else {
#pragma unroll
                    for (int c4 = 0; c4 < 3; ++c4)
                        asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};"
                                     ::"r"(xq + uint32_t(3 * (dy >> 1) + c4) * (kFR * kFC * 16) + pix * 16u), "f"(Qd[4 * c4]), "f"(Qd[4 * c4 + 1]),
                                       "f"(Qd[4 * c4 + 2]), "f"(Qd[4 * c4 + 3]) : "memory");
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(F_DEMPTY + g));                  // accumulator g may be overwritten
            asm volatile("bar.sync 1, 384;" ::: "memory");                 // the 12 row warps
            const int y = t.y0 + r, x = t.x0 + cx;
            if (r >= 1 && r <= kFOutR && cx >= 1 && cx <= kFOutC && y < p.H && x < p.W) {
                float o[12];
#pragma unroll
                for (int c4 = 0; c4 < 3; ++c4) {
                    float4 up, dn;                                         // Q[0] of row r-1, Q[2] of row r+1
                    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(up.x), "=f"(up.y), "=f"(up.z), "=f"(up.w)
                                 : "r"(xq + uint32_t(c4) * (kFR * kFC * 16) + (pix - kFC) * 16u));
                    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(dn.x), "=f"(dn.y), "=f"(dn.z), "=f"(dn.w)
                                 : "r"(xq + uint32_t(3 + c4) * (kFR * kFC * 16) + (pix + kFC) * 16u));
                    o[4 * c4 + 0] = bs[4 * c4 + 0] + up.x + Q1[4 * c4 + 0] + dn.x;
                    o[4 * c4 + 1] = bs[4 * c4 + 1] + up.y + Q1[4 * c4 + 1] + dn.y;
                    o[4 * c4 + 2] = bs[4 * c4 + 2] + up.z + Q1[4 * c4 + 2] + dn.z;
                    o[4 * c4 + 3] = bs[4 * c4 + 3] + up.w + Q1[4 * c4 + 3] + dn.w;
                }
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
    if (!tc_encode_3d(&m.tm_w, L.w, 64, kFN, (unsigned long long)L.groups, 64, kFN, 1, err)) return false;
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
    p.groups = L.groups;
    p.bias = L.bias;
    p.out = out; p.out_h = out_h; p.out_w = out_w;
    const int grid = p.total_tiles < num_sms ? p.total_tiles : num_sms;
    return launch_pdl(final_is_kernel, grid, kFThreads, kFSmem, st, 1, m.tm_in, m.tm_w, p);
}

}  // namespace ufnvc
