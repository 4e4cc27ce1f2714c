// CUDA-core implicit-GEMM convolution (any channel count that is a multiple of 8) and the depthwise 3x3.
// The generic conv serves the shapes the tcgen05 kernel does not take (config 1's 48/32/16-channel layers) and is
// the on-device cross-check of the tensor-core path.  Activations NHWC bf16, fp32 accumulate.
//   out[pix][n] = bias[n] + sum_{tap, c} in[pix + tap][c] * w[group][tap][n][c]
#include "epilogue.cuh"
#include "tc_ptx.cuh"
#include "ufnvc_internal.h"

namespace ufnvc {

constexpr int GM = 64, GN = 64, GK = 32;

__global__ void __launch_bounds__(256) conv_generic_kernel(const bf16 *__restrict__ in, const bf16 *__restrict__ wt,
                                                           const float *__restrict__ bias, int n_img, int H, int W,
                                                           int c_in, int n_real, int n_pad, int taps, int groups,
                                                           EpiParams E)
{
    __shared__ float As[GK][GM + 4];
    __shared__ float Bs[GK][GN + 4];
    const int img = blockIdx.z;
    const int grp = groups == 1 ? 0 : img % groups;
    const int P = H * W;
    const int m0 = blockIdx.x * GM, n0 = blockIdx.y * GN;
    const int tid = threadIdx.x, ty = tid / 16, tx = tid % 16;

    // loaders: 64 rows x 32 k, 8 consecutive k (16 bytes) per thread
    const int l_row = tid / 4, l_k = (tid % 4) * 8;
    const int pm = m0 + l_row;
    const int py = pm < P ? pm / W : 0, px = pm < P ? pm % W : 0;
    const bf16 *in_img = in + (long long)img * P * c_in;
    const bf16 *w_grp = wt + (long long)grp * taps * n_pad * c_in;

    float acc[4][4] = {};
    for (int tap = 0; tap < taps; ++tap) {
        const int dy = taps == 9 ? tap / 3 - 1 : 0, dx = taps == 9 ? tap % 3 - 1 : 0;
        const int yy = py + dy, xx = px + dx;
        const bool a_ok = pm < P && yy >= 0 && yy < H && xx >= 0 && xx < W;
        const bf16 *a_src = in_img + ((long long)yy * W + xx) * c_in;
        const bool b_ok = n0 + l_row < n_pad;
        const bf16 *b_src = w_grp + ((long long)tap * n_pad + n0 + l_row) * c_in;
        for (int k0 = 0; k0 < c_in; k0 += GK) {
            uint4 av = make_uint4(0, 0, 0, 0), bv = make_uint4(0, 0, 0, 0);
            if (k0 + l_k < c_in) {
                if (a_ok) av = *reinterpret_cast<const uint4 *>(a_src + k0 + l_k);
                if (b_ok) bv = *reinterpret_cast<const uint4 *>(b_src + k0 + l_k);
            }
            const bf16 *ae = reinterpret_cast<const bf16 *>(&av), *be = reinterpret_cast<const bf16 *>(&bv);
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                As[l_k + e][l_row] = __bfloat162float(ae[e]);
                Bs[l_k + e][l_row] = __bfloat162float(be[e]);
            }
            __syncthreads();
#pragma unroll
            for (int k = 0; k < GK; ++k) {
                const float4 a4 = *reinterpret_cast<const float4 *>(&As[k][ty * 4]);
                const float4 b4 = *reinterpret_cast<const float4 *>(&Bs[k][tx * 4]);
                const float a[4] = {a4.x, a4.y, a4.z, a4.w}, b[4] = {b4.x, b4.y, b4.z, b4.w};
#pragma unroll
                for (int i = 0; i < 4; ++i)
#pragma unroll
                    for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
            }
            __syncthreads();
        }
    }

    const float *b_grp = bias + (long long)grp * n_pad;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int m = m0 + ty * 4 + i;
        if (m >= P) continue;
        const int y = m / W, x = m % W;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int n = n0 + tx * 4 + j;
            if (n >= n_real) continue;
            float v = apply_act(acc[i][j] + b_grp[n], E.act);
            if (E.mode == EPI_FINAL) {
                epi_store_final(E, img, y, x, n, v);
            } else {
                const long long o = epi_offset(E, img, y, x, H, W, n);
                if (E.residual) v += __bfloat162float(E.residual[o]);
                reinterpret_cast<bf16 *>(E.out)[o] = __float2bfloat16_rn(v);
            }
        }
    }
}

cudaError_t launch_conv_generic(const ConvLayer &L, const ConvProblem &P, const EpiParams &E, LaunchStream st)
{
    dim3 grid((P.H * P.W + GM - 1) / GM, (L.n + GN - 1) / GN, P.n_img);
    conv_generic_kernel<<<grid, 256, 0, st>>>(P.in, L.w, L.bias, P.n_img, P.H, P.W, L.c_in, L.n, L.n_pad, L.taps, L.groups, E);
    return cudaGetLastError();
}

// ---- A6: depthwise 3x3, zero pad, bias.  HBM-bound.  A thread owns 8 channels (one 16-byte vector)
// of one pixel column x and walks down a segment of rows: each input row is loaded once as 3 vectors (x-1, x, x+1;
// the side columns are L1 hits, loaded by the neighbouring warps of the block) and scattered into three rolling
// accumulators (output rows r-1, r, r+1), so a row of outputs costs 3 vector loads and 1 store.  For C = 256 a warp is
// exactly one pixel (512 contiguous bytes).
// bf16x2 word -> packed (lo, hi) fp32 pair for the FFMA2 pipe: 2 integer ops.  The shift is written as a byte permute so
// that it issues on the ALU pipe: the compiler turns "w << 16" into IMAD.U32, which competes with FFMA2 for the FMA pipe.
__device__ __forceinline__ uint64_t dw_pair(uint32_t w)
{
    uint32_t lo;
    asm("prmt.b32 %0, %1, 0, 0x1044;" : "=r"(lo) : "r"(w));
    return f2_pack(__uint_as_float(lo), __uint_as_float(w & 0xFFFF0000u));
}

__global__ void __launch_bounds__(256, 2) dwconv3x3_kernel(const bf16 *__restrict__ in, bf16 *__restrict__ out,
                                                        const float *__restrict__ w9c, const float *__restrict__ bias,
                                                        int n_img, int H, int W, int C, int rows_per_seg, int n_seg)
{
    const int cv = C / 8;
    const long long total = (long long)n_img * n_seg * W * cv;
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= total) return;
    const int c8 = int(t % cv);
    long long r = t / cv;
    const int x = int(r % W); r /= W;
    const int seg = int(r % n_seg);
    const int img = int(r / n_seg);
    const int c0 = c8 * 8;
    const int y0 = seg * rows_per_seg, y1 = min(H, y0 + rows_per_seg);      // output rows [y0, y1)

    uint64_t wv[9][4], bv[4];                                               // channel pairs (2e, 2e+1)
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        const float4 lo = __ldg(reinterpret_cast<const float4 *>(w9c + k * C + c0));
        const float4 hi = __ldg(reinterpret_cast<const float4 *>(w9c + k * C + c0 + 4));
        wv[k][0] = f2_pack(lo.x, lo.y); wv[k][1] = f2_pack(lo.z, lo.w);
        wv[k][2] = f2_pack(hi.x, hi.y); wv[k][3] = f2_pack(hi.z, hi.w);
    }
    {
        const float4 lo = __ldg(reinterpret_cast<const float4 *>(bias + c0)), hi = __ldg(reinterpret_cast<const float4 *>(bias + c0 + 4));
        bv[0] = f2_pack(lo.x, lo.y); bv[1] = f2_pack(lo.z, lo.w); bv[2] = f2_pack(hi.x, hi.y); bv[3] = f2_pack(hi.z, hi.w);
    }
    const bf16 *img_in = in + (long long)img * H * W * C + c0;
    bf16 *img_out = out + (long long)img * H * W * C + c0;
    const bool has_l = x > 0, has_r = x + 1 < W;
    const uint4 z4 = make_uint4(0, 0, 0, 0);
    auto load_row = [&](int ir, uint4 &vl, uint4 &vc, uint4 &vr) {
        vl = vc = vr = z4;
        if (ir >= 0 && ir < H && ir <= y1) {
            const bf16 *row = img_in + ((long long)ir * W + x) * C;
            if (has_l) vl = __ldg(reinterpret_cast<const uint4 *>(row - C));
            vc = __ldg(reinterpret_cast<const uint4 *>(row));
            if (has_r) vr = __ldg(reinterpret_cast<const uint4 *>(row + C));
        }
    };

    uint64_t accP[4], accC[4], accN[4];         // outputs rows ir-1, ir, ir+1 while input row ir is being added
#pragma unroll
    for (int e = 0; e < 4; ++e) { accP[e] = bv[e]; accC[e] = bv[e]; accN[e] = bv[e]; }

    uint4 nl, nc, nr;
    load_row(y0 - 1, nl, nc, nr);
    for (int ir = y0 - 1; ir <= y1; ++ir) {     // input rows feeding outputs [y0, y1); rows outside the image are zeros
        const uint4 vl = nl, vc = nc, vr = nr;
        load_row(ir + 1, nl, nc, nr);           // next row's loads are in flight while this row is accumulated
        const uint32_t *pl = reinterpret_cast<const uint32_t *>(&vl), *pc = reinterpret_cast<const uint32_t *>(&vc),
                       *pr = reinterpret_cast<const uint32_t *>(&vr);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const uint64_t fl = dw_pair(pl[e]), fc = dw_pair(pc[e]), fr = dw_pair(pr[e]);
            // input row ir is kernel row 2 of output ir-1, row 1 of output ir, row 0 of output ir+1
            accP[e] = f2_fma(wv[6][e], fl, f2_fma(wv[7][e], fc, f2_fma(wv[8][e], fr, accP[e])));
            accC[e] = f2_fma(wv[3][e], fl, f2_fma(wv[4][e], fc, f2_fma(wv[5][e], fr, accC[e])));
            accN[e] = f2_fma(wv[0][e], fl, f2_fma(wv[1][e], fc, f2_fma(wv[2][e], fr, accN[e])));
        }
        const int oy = ir - 1;                  // output row oy is complete once input row oy+1 = ir has been added
        if (oy >= y0 && oy < y1) {
            uint4 o;
            __nv_bfloat162 *oe = reinterpret_cast<__nv_bfloat162 *>(&o);
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                float a, b;
                f2_unpack(accP[e], a, b);
                oe[e] = __floats2bfloat162_rn(a, b);
            }
            *reinterpret_cast<uint4 *>(img_out + ((long long)oy * W + x) * C) = o;
        }
#pragma unroll
        for (int e = 0; e < 4; ++e) { accP[e] = accC[e]; accC[e] = accN[e]; accN[e] = bv[e]; }
    }
}

// ---- A6, TMA-staged kernel (C a multiple of 64).  One tile = 8 x 8 pixels of one image, all channels: one TMA box
// {64 ch, 10, 10} per 64-channel slab brings the tile plus halo into shared memory (zero-filled outside the image =
// the conv's zero padding).  The kernel is persistent (two blocks per SM) and double-buffered: the load of a block's
// next tile is in flight while it computes the current one, so ~100 KB per block are in flight without costing a
// register -- the register-only kernel above is latency-bound (16 warps/SM, 8 KB of unique loads in flight).
constexpr int kDwT = 8;                                   // tile edge (pixels)
constexpr int kDwHalo = kDwT + 2;
constexpr uint32_t kDwSlab = ((kDwHalo * kDwHalo * 128 + 1023) / 1024) * 1024;     // 13312 B per 64-channel slab (dense box, no swizzle)

// Column-blocked: a thread owns ONE channel pair of NC adjacent columns (a first version gave it four pairs of one column): a warp is the 32 pairs of one 64-channel slab,
// so a halo pixel is one conflict-free LDS.32 wavefront (128 contiguous bytes), a halo row of NC + 2 pixels serves NC
// outputs (NC + 2 bf16x2 -> f32x2 conversions instead of 3 NC), the 9 weights take 18 registers instead of 72 and the bias
// stays in registers.  ncu on the 8-channel kernel showed why this matters: nothing saturated (issue 44 %, FMA 21 %, ALU
// 30 %), 4 warps per scheduler at 128 registers, 0.83 eligible.  Bottom-edge tiles stop at the last image row and are
// ordered last, so the blocks that get one tile more than the others get the cheap ones.
constexpr int kDwNC = 4;                                 // columns per thread
// Warp roles: CC / 32 compute warps and one producer warp.  The producer claims tiles (a per-launch counter if given, else
// static striding), waits for their inputs, and issues their TMA as soon as the buffer is free; compute warps only ever wait on
// the full barrier of their buffer and release it with one arrive per warp -- no block-wide barrier per tile.
template <int CC>                                         // CC = channel count (64, 128, 192 or 256), compile-time so that the
__global__ void __launch_bounds__(CC + 32, 2) dwconv3x3_cols_kernel(const __grid_constant__ CUtensorMap tm_in, bf16 *__restrict__ out,  // column
                                                             const float *__restrict__ w9c, const float *__restrict__ bias,     // stores are
                                                             int n_img, int H, int W, int tiles_x, int tiles_y,                 // immediates
                                                             uint32_t *__restrict__ sched, const uint32_t *dep_flags, uint32_t dep_need)
{
    constexpr int NC = kDwNC, C = CC, slabs = CC >> 6;
    extern __shared__ __align__(1024) uint8_t dw_smem[];
    const uint32_t base = (smem_u32(dw_smem) + 1023u) & ~1023u;
    constexpr uint32_t buf_bytes = uint32_t(slabs) * kDwSlab;
    const uint32_t bar = base + 2u * buf_bytes;                       // full[0], full[1], empty[0], empty[1]
    volatile int *s_tile = reinterpret_cast<volatile int *>(dw_smem + (bar + 32u - smem_u32(dw_smem)));   // tile held by each buffer, -1 = none
    const int n_tiles = n_img * tiles_x * tiles_y;
    const int n_full = n_img * tiles_x * (tiles_y - 1);               // tiles above the bottom tile row come first
    auto coord = [&](int t, int &tx, int &ty, int &im) {
        if (t < n_full) {
            tx = t % tiles_x;
            const int r = t / tiles_x;
            ty = r % (tiles_y - 1); im = r / (tiles_y - 1);
        } else {
            const int u = t - n_full;
            tx = u % tiles_x; im = u / tiles_x; ty = tiles_y - 1;
        }
    };
    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        mbar_init(bar + 8, 1);
        mbar_init(bar + 16, CC / 32);
        mbar_init(bar + 24, CC / 32);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    const int lane = threadIdx.x & 31;
    __syncthreads();                                                  // barriers initialised before anyone touches them

    if (threadIdx.x >= CC) {
        // ===================== producer warp =====================
        // The input is the predecessor's output.  Without dep_flags the whole predecessor grid is waited for (PDL).  With
        // dep_flags (tail filling) the predecessor is the trunk MLP kernel of the previous block, which counts its finished
        // 128-pixel tiles: a tile of this kernel then only waits for the MLP tiles that cover its halo box, so the blocks of
        // this grid that become resident while the MLP kernel runs its last, partly filled round start working.  Those MLP
        // tiles have also finished READING the rows of `out` this tile overwrites (an MLP tile reads its rows of `out`, this
        // kernel's output buffer, before it writes and counts), and every older kernel completed before the MLP kernel passed
        // its own griddepcontrol.wait, which precedes the launch of this grid.
        if (!dep_flags) asm volatile("griddepcontrol.wait;" ::: "memory");
        asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
        for (uint32_t it = 0;; ++it) {
            const uint32_t b = it & 1u;
            int t = int(blockIdx.x + it * gridDim.x);
            if (sched) {
                if (lane == 0) t = int(atomicAdd(sched, 1u));
                t = __shfl_sync(0xFFFFFFFFu, t, 0);
            }
            if (t >= n_tiles) t = -1;
            int tx = 0, ty = 0, im = 0;
            if (t >= 0) coord(t, tx, ty, im);
            if (t >= 0 && dep_flags) {
                const int ya = max(ty * kDwT - 1, 0), yb = min(ty * kDwT + kDwT, H - 1);
                const int xa = max(tx * kDwT - 1, 0), xb = min(tx * kDwT + kDwT, W - 1);
                const int f_lo = int((((long long)im * H + ya) * W + xa) >> 7), f_hi = int((((long long)im * H + yb) * W + xb) >> 7);
                for (int f = f_lo + lane; f <= f_hi; f += 32) {
                    uint32_t v, spins = 0;
                    for (;;) {
                        asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(dep_flags + f) : "memory");
                        if (v >= dep_need) break;
                        __nanosleep(64);
                        if (++spins > (1u << 22)) __trap();            // seconds: the producer kernel is gone; fail loudly, never hang
                    }
                }
                asm volatile("fence.acq_rel.gpu;" ::: "memory");
                __syncwarp();
            }
            if (it >= 2) mbar_wait(bar + 16u + 8u * b, ((it >> 1) - 1u) & 1u);    // every compute warp has released buffer b
            if (elect_one()) {
                s_tile[b] = t;
                if (t < 0) {
                    mbar_arrive(bar + 8u * b);                        // completes the phase: the compute warps read -1 and leave
                } else {
                    if (dep_flags) asm volatile("fence.proxy.async;" ::: "memory");   // the MLP kernel's generic-proxy writes -> this TMA read
                    mbar_expect_tx(bar + 8u * b, uint32_t(slabs) * (kDwHalo * kDwHalo * 128));
#pragma unroll
                    for (int s = 0; s < slabs; ++s)
                        tma_load_4d(base + b * buf_bytes + uint32_t(s) * kDwSlab, &tm_in, bar + 8u * b, s * 64, tx * kDwT - 1, ty * kDwT - 1, im);
                }
            }
            __syncwarp();
            if (t < 0) break;
        }
        return;
    }

    // ===================== compute warps =====================
    constexpr int cp = C >> 1;                                        // channel pairs; a multiple of 32
    const int g = threadIdx.x / cp, p = threadIdx.x % cp;             // column group of the tile, channel pair
    const int c0 = 2 * p;
    uint64_t wv[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) {                                     // weights and bias are static: no wait needed
        const float2 q = __ldg(reinterpret_cast<const float2 *>(w9c + k * C + c0));
        wv[k] = f2_pack(q.x, q.y);
    }
    uint64_t bv;
    {
        const float2 q = __ldg(reinterpret_cast<const float2 *>(bias + c0));
        bv = f2_pack(q.x, q.y);
    }
    const long long row_stride = (long long)W * C;
    for (uint32_t it = 0;; ++it) {
        const uint32_t b = it & 1u;
        mbar_wait(bar + 8u * b, (it >> 1) & 1u);
        const int tile = s_tile[b];                                   // written by the producer before its arrive on full[b]
        if (tile < 0) break;
        int tx, ty, img;
        coord(tile, tx, ty, img);
        const int x0 = tx * kDwT + g * NC, y0 = ty * kDwT;
        const int n_cols = W - x0;                                    // columns j < n_cols are inside the image
        // halo pixel (hy, g * NC + j), this thread's pair: lanes of a warp read 128 contiguous bytes
        const uint32_t tb = base + b * buf_bytes + uint32_t(p >> 5) * kDwSlab + uint32_t(p & 31) * 4u + uint32_t(g * NC) * 128u;
        uint64_t accP[NC], accC[NC], accN[NC];
#pragma unroll
        for (int j = 0; j < NC; ++j) { accP[j] = 0ull; accC[j] = 0ull; accN[j] = 0ull; }
        bf16 *dst = out + (((long long)img * H + y0) * W + x0) * C + c0;
#pragma unroll
        for (int hy = 0; hy < kDwHalo; ++hy) {                        // halo row hy = image row y0 - 1 + hy
            if (hy >= 3 && y0 + hy - 2 >= H) break;                   // block-uniform: no output row needs this halo row
            uint64_t f[NC + 2];
#pragma unroll
            for (int j = 0; j < NC + 2; ++j) {
                uint32_t w;
                asm volatile("ld.shared.b32 %0, [%1];" : "=r"(w) : "r"(tb + uint32_t(hy * kDwHalo + j) * 128u));
                f[j] = dw_pair(w);
            }
#pragma unroll
            for (int j = 0; j < NC; ++j) {
                accP[j] = f2_fma(wv[6], f[j], f2_fma(wv[7], f[j + 1], f2_fma(wv[8], f[j + 2], accP[j])));
                accC[j] = f2_fma(wv[3], f[j], f2_fma(wv[4], f[j + 1], f2_fma(wv[5], f[j + 2], accC[j])));
                accN[j] = f2_fma(wv[0], f[j], f2_fma(wv[1], f[j + 1], f2_mul(wv[2], f[j + 2])));
            }
            if (hy >= 2) {                                            // output row y0 + hy - 2 is complete
                __nv_bfloat162 o[NC];
#pragma unroll
                for (int j = 0; j < NC; ++j) {
                    float a, b2;
                    f2_unpack(f2_add(accP[j], bv), a, b2);
                    o[j] = __floats2bfloat162_rn(a, b2);
                }
#pragma unroll
                for (int j = 0; j < NC; ++j)                          // predicated stores at immediate offsets j * C
                    if (j < n_cols) *reinterpret_cast<__nv_bfloat162 *>(dst + j * C) = o[j];
                dst += row_stride;
            }
#pragma unroll
            for (int j = 0; j < NC; ++j) { accP[j] = accC[j]; accC[j] = accN[j]; }
        }
        __syncwarp();                                                 // every lane of this warp is done reading buffer b
        if (lane == 0) mbar_arrive(bar + 16u + 8u * b);
    }
}

template <int CC>
static cudaError_t launch_dw_cols(const CUtensorMap &tm_in, bf16 *out, const float *w9c, const float *bias, int n_img, int H, int W,
                                  int tiles_x, int tiles_y, int grid, size_t smem, LaunchStream st, uint32_t *sched, const uint32_t *dep)
{
    return launch_pdl(dwconv3x3_cols_kernel<CC>, grid, CC + 32, smem, st, 1, tm_in, out, w9c, bias, n_img, H, W, tiles_x, tiles_y, sched, dep, kTrunkTileSignals);
}

cudaError_t configure_depthwise_kernels()
{
    cudaError_t e = cudaFuncSetAttribute(dwconv3x3_cols_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(dwconv3x3_cols_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(dwconv3x3_cols_kernel<192>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(dwconv3x3_cols_kernel<256>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    return e;
}

cudaError_t launch_dwconv3x3_tma(const CUtensorMap &tm_in, bf16 *out, const float *w9c, const float *bias, int n_img, int H, int W,
                                 int C, int num_sms, LaunchStream st, uint32_t *sched, const uint32_t *dep_flags)
{
    const int tiles_x = (W + kDwT - 1) / kDwT, tiles_y = (H + kDwT - 1) / kDwT;
    const size_t smem = 1024 + 2 * size_t(C >> 6) * kDwSlab + 48;     // + four barriers + the two tile slots
    const int n_tiles = n_img * tiles_x * tiles_y;
    const int grid = n_tiles < 2 * num_sms ? n_tiles : 2 * num_sms;    // persistent: two blocks per SM, double-buffered tiles
    switch (C) {
        case 64: return launch_dw_cols<64>(tm_in, out, w9c, bias, n_img, H, W, tiles_x, tiles_y, grid, smem, st, sched, dep_flags);
        case 128: return launch_dw_cols<128>(tm_in, out, w9c, bias, n_img, H, W, tiles_x, tiles_y, grid, smem, st, sched, dep_flags);
        case 192: return launch_dw_cols<192>(tm_in, out, w9c, bias, n_img, H, W, tiles_x, tiles_y, grid, smem, st, sched, dep_flags);
        case 256: return launch_dw_cols<256>(tm_in, out, w9c, bias, n_img, H, W, tiles_x, tiles_y, grid, smem, st, sched, dep_flags);
        default: return cudaErrorInvalidValue;
    }
}

cudaError_t launch_dwconv3x3(const bf16 *in, bf16 *out, const float *w9c, const float *bias, int n_img, int H, int W,
                             int C, LaunchStream st)
{
    // segment length: the shortest of {H, 16, 8} rows that still gives >= ~32 warps per SM (148 SMs)
    int rows = H;
    const long long per_row_threads = (long long)n_img * W * (C / 8);
    while (rows > 8 && per_row_threads * ((H + rows - 1) / rows) < 148LL * 32 * 32) rows = (rows + 1) / 2;
    const int n_seg = (H + rows - 1) / rows;
    const long long total = per_row_threads * n_seg;
    dwconv3x3_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(in, out, w9c, bias, n_img, H, W, C, rows, n_seg);
    return cudaGetLastError();
}

}  // namespace ufnvc
