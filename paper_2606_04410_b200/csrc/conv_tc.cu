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
#include "tc_ptx.cuh"
#include "ufnvc_internal.h"

namespace ufnvc {

namespace {

constexpr int kStages = 4;
constexpr int kTileM = 128;
constexpr int kSlabK = 64;                       // bf16 channels per smem row = 128 bytes = one swizzle span
constexpr int kABytes = kTileM * kSlabK * 2;     // 16 KB
constexpr int kThreads = 320;                    // warp 0 TMA, warp 1 MMA, warps 2..9 epilogue

// n / d for 0 <= n < 2^31 as one multiply-high, one add and one shift (Granlund-Montgomery round-up method): the
// per-tile index arithmetic sits on the single-thread MMA-issue path, where a hardware-emulated division costs ~40
// dependent instructions.
struct FastDiv {
    uint32_t d, mul, shr;
    __device__ __forceinline__ uint32_t div(uint32_t n) const { return (__umulhi(n, mul) + n) >> shr; }
    __device__ __forceinline__ void divmod(uint32_t n, uint32_t &q, uint32_t &r) const { q = div(n); r = n - q * d; }
};
static FastDiv make_fastdiv(uint32_t d)
{
    FastDiv f;
    f.d = d;
    uint32_t l = 0;
    while ((1ull << l) < d) ++l;
    f.mul = uint32_t(((1ull << 32) * ((1ull << l) - d)) / d + 1);
    f.shr = l;
    return f;
}

struct TcParams {
    FastDiv fd_ntiles, fd_tx, fd_ty, fd_groups;
    int n_img_m, Hm, Wm;          // activation as the TMA map sees it (flattened for 1x1 convs)
    int flat, tw_shift;           // flat: rows of 128 consecutive pixels; tw_shift = log2(TW)
    int tiles_y, tiles_x, TH, TW;
    int xpose;                    // CTA-pair halo kernel: the map's dimension 1 is the image's y and dimension 2 its x (Hm = W, Wm = H)
    int tiles_img;                // CTA-pair halo kernel: tiles per image; the schedule runs over PAIRS of consecutive tiles
    int reverse;                  // CTA-pair halo kernel: schedule unit u stands for unit total_tiles - 1 - u
    FastDiv fd_pairs;             // pairs per image = ceil(tiles_img / 2)
    int H, W;                     // real image dims: global pixel -> (img, y, x) for the epilogue
    int taps, slabs;              // k-blocks per tile = taps * slabs
    int tap_img;                  // 1: tap t is image img * taps + t of the activation map (fold over stacked images), no spatial shift
    int n_tiles, BN, n_real, n_pad;
    int groups;
    int total_tiles;
    const float *bias;            // [groups][n_pad]
    EpiParams E;
};

}  // namespace

namespace {

// tile index -> (image in map space, tile origin, n tile); n fastest so CTAs running side by side share the A tile in L2
struct TileCoord { int img, y0, x0, nt; };
__device__ __forceinline__ int group_of(const TcParams &p, int img)
{
    if (p.groups == 1) return 0;
    uint32_t q, r;
    p.fd_groups.divmod(uint32_t(img), q, r);
    return int(r);
}
__device__ __forceinline__ TileCoord tile_coord(const TcParams &p, int tile)
{
    TileCoord c;
    uint32_t r, nt, tx, ty, img;
    p.fd_ntiles.divmod(uint32_t(tile), r, nt);
    p.fd_tx.divmod(r, r, tx);
    p.fd_ty.divmod(r, img, ty);
    c.nt = int(nt);
    c.img = int(img);
    c.y0 = int(ty) * p.TH;
    c.x0 = int(tx) * p.TW;
    return c;
}

// CTA-pair halo kernel: schedule unit -> this CTA's tile.  A unit is (image, pair of consecutive tiles of that image in row-major
// tile order, n tile); the two tiles of a pair need not be neighbours (each CTA loads its own halo box, the pair shares only the
// weights), so an odd tile count per row costs nothing and only an odd count per IMAGE leaves one half-empty pair.  A tile past
// the image's last gets an origin outside the map: TMA fills zeros and the epilogue's bounds test masks it.
__device__ __forceinline__ TileCoord tile_coord_pair(const TcParams &p, int unit, int rank)
{
    TileCoord c;
    uint32_t r, nt, pi, img, ty, tx;
    if (p.reverse) unit = p.total_tiles - 1 - unit;
    p.fd_ntiles.divmod(uint32_t(unit), r, nt);
    p.fd_pairs.divmod(r, img, pi);
    const uint32_t id = 2 * pi + uint32_t(rank);
    p.fd_tx.divmod(id, ty, tx);
    c.nt = int(nt);
    c.img = int(img);
    c.y0 = int(id) < p.tiles_img ? int(ty) * p.TH : p.Hm + p.TH;
    c.x0 = int(tx) * p.TW;
    return c;
}

// 8 epilogue warps: warp w reads TMEM lanes 32*(w%4) .. +31 (a hardware rule), and the two warps of a lane quadrant
// split the 32-column chunks between them (even / odd), so every SM sub-partition holds two epilogue warps and the
// tcgen05.ld / MUFU latencies of one hide behind the other.  tcgen05.ld -> bias -> act -> store, per tile of the
// persistent schedule; tfull0 / tempty0 are the smem addresses of the first of two consecutive mbarriers each.
// pair_rank >= 0: CTA-pair kernel -- the schedule runs over tile PAIRS (blockIdx.x / 2, stride gridDim.x / 2), this CTA
// owns x tile 2 * txp + pair_rank, and tempty0 is the LEADER's barrier as a cluster address (relaxed remote arrive).
template <int MODE>
__device__ __forceinline__ void epilogue_warps(const TcParams &p, uint32_t tmem_base, uint32_t tfull0, uint32_t tempty0,
                                               int warp, int lane, int pair_rank = -1)
{
    const int quad = warp & 3;
    const int half = (warp - 2) >> 2;                             // 0: even 32-column chunks, 1: odd ones
    const int m = quad * 32 + lane;                               // accumulator row = pixel inside the tile
    const int my = m >> p.tw_shift, mx = m & (p.TW - 1);          // TW is a power of two
    const unsigned P = unsigned(p.H) * unsigned(p.W);
    int it = 0;
    const int tile0 = pair_rank < 0 ? int(blockIdx.x) : int(blockIdx.x >> 1), tstride = pair_rank < 0 ? int(gridDim.x) : int(gridDim.x >> 1);
    for (int tile = tile0; tile < p.total_tiles; tile += tstride, ++it) {
        const TileCoord tc = pair_rank >= 0 ? tile_coord_pair(p, tile, pair_rank) : tile_coord(p, tile);
        const int acc = it & 1;
        const uint32_t acc_phase = (it >> 1) & 1;
        const int ym = tc.y0 + my, xm = tc.x0 + mx;
        const bool inb = ym < p.Hm && xm < p.Wm;
        int img = tc.img, y = ym, x = xm;
        if (p.xpose) { y = xm; x = ym; }                          // transposed tile map: map dimension 1 is the image's y
        if (p.flat) {                                             // map-space row of 128 pixels -> real (img, y, x)
            const unsigned gp = unsigned(ym) * 128u + unsigned(xm);
            img = int(gp / P);
            const unsigned rem = gp - unsigned(img) * P;
            y = int(rem / unsigned(p.W));
            x = int(rem - unsigned(y) * unsigned(p.W));
        }
        const int grp = group_of(p, img);
        const float *bias = p.bias + (long long)grp * p.n_pad + tc.nt * p.BN;
        float bias_lane[4] = {0.f, 0.f, 0.f, 0.f};                   // EPI_HEAD: bias of column c0 + lane for this warp's chunks
        float wn_lane[4] = {0.f, 0.f, 0.f, 0.f};                     // EPI_HEAD: kappa_t * |w row|_2 of the same columns
        float xpatch = 0.f;                                          // EPI_HEAD: |x|_2 over the 3x3 neighbourhood of this z-pixel
        if (MODE == EPI_HEAD) {
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if (half * 32 + q * 64 < p.BN) {
                    bias_lane[q] = __ldg(bias + half * 32 + q * 64 + lane);
                    wn_lane[q] = p.E.kappa_t * __ldg(p.E.wnorm + tc.nt * p.BN + half * 32 + q * 64 + lane);
                }
            if (inb) {
                float s2 = 0.f;
#pragma unroll
                for (int t = 0; t < 9; ++t) {
                    const int yy = y + t / 3 - 1, xx = x + t % 3 - 1;
                    if (yy >= 0 && yy < p.H && xx >= 0 && xx < p.W) {
                        const float *xp = p.E.xnorm2 + (((long long)img * p.H + yy) * p.W + xx) * p.E.xnorm_parts;
                        for (int q = 0; q < p.E.xnorm_parts; ++q) s2 += __ldg(xp + q);
                    }
                }
                xpatch = sqrtf(s2);
            }
        }
        mbar_wait(tfull0 + 8u * acc, acc_phase);
        tc_fence_after();
        const uint32_t t_row = tmem_base + (uint32_t(quad * 32) << 16) + uint32_t(acc * p.BN);
        if (MODE == EPI_FINAL) {
            if (half == 0) {
                uint32_t v[16];
                tmem_ld16(t_row, v);
                if (inb) {
                    if (p.E.c_o == 3 && p.n_real == 12 && !(p.E.out_w & 1)) {
                        // packed column n = (2i + j) * 3 + c -> out[img][c][2y + i][2x + j]: j = 0, 1 are one float2
                        float *base = reinterpret_cast<float *>(p.E.out) + (long long)img * p.E.img_stride;
                        const int ox = 2 * x;
                        if (ox < p.E.out_w) {
#pragma unroll
                            for (int i = 0; i < 2; ++i) {
                                const int oy = 2 * y + i;
                                if (oy >= p.E.out_h) continue;
#pragma unroll
                                for (int c = 0; c < 3; ++c) {
                                    const int n0 = (2 * i) * 3 + c, n1 = (2 * i + 1) * 3 + c;
                                    float2 o2;
                                    o2.x = fminf(fmaxf(__uint_as_float(v[n0]) + __ldg(bias + n0), 0.0f), 1.0f);
                                    o2.y = fminf(fmaxf(__uint_as_float(v[n1]) + __ldg(bias + n1), 0.0f), 1.0f);
                                    *reinterpret_cast<float2 *>(base + ((long long)c * p.E.out_h + oy) * p.E.out_w + ox) = o2;
                                }
                            }
                        }
                    } else {
#pragma unroll
                        for (int j = 0; j < 16; ++j) {
                            const int n = tc.nt * p.BN + j;
                            if (n < p.n_real) epi_store_final(p.E, img, y, x, n, __uint_as_float(v[j]) + __ldg(bias + j));
                        }
                    }
                }
            }
        } else if (MODE == EPI_HEAD) {
            // A2: pixel-shuffle x4 + crop + split.  A 32-column chunk is 32 consecutive latent channels of one sub-pixel.
            // The map is tiny (one tile per CTA), so nothing overlaps this epilogue and its serial latencies are the
            // cost: the biases are read BEFORE the accumulator is waited for (one per lane and chunk, handed round by
            // shuffles), and the list-slot atomic of a chunk is consumed one chunk later.
            const EpiParams &E = p.E;
            uint32_t pend_fm = 0, pend_off = 0, pend_base = 0, pend_total = 0;
            long long pend_e0 = 0;
            auto flush_pending = [&]() {
                if (pend_total) {                                               // warp-uniform
                    uint32_t w = __shfl_sync(0xFFFFFFFFu, pend_base, 31) + pend_off;
                    while (pend_fm) {
                        const int j = __ffs(pend_fm) - 1;
                        pend_fm &= pend_fm - 1;
                        E.fix_list[w++] = uint32_t(pend_e0 + j);
                    }
                }
                pend_total = 0;
            };
            for (int c0 = half * 32; c0 < p.BN; c0 += 64) {
                uint32_t v[32];
                tmem_ld32(t_row + uint32_t(c0), v);
                const float bl = bias_lane[c0 >> 6], wl = wn_lane[c0 >> 6];
                const int n = tc.nt * p.BN + c0;
                const int sij = n / E.c_y, c2 = n - sij * E.c_y;
                const int ly = 4 * y + ((sij >> 2) & 3), lx = 4 * x + (sij & 3);
                const bool live = inb && ly < E.lat_h && lx < E.lat_w;             // crop [R2]; dead lanes still join the scans
                const long long e0 = (((long long)img * E.lat_h + ly) * E.lat_w + lx) * E.c_y + c2;
                float f[32];
#pragma unroll
                for (int j = 0; j < 32; ++j) f[j] = __uint_as_float(v[j]) + __shfl_sync(0xFFFFFFFFu, bl, j);
                if ((sij >> 4) == 0) {                                             // mean (n is warp-uniform)
                    if (live) {
#pragma unroll
                        for (int q = 0; q < 4; ++q) st_global_256(E.mu + e0 + 8 * q, f + 8 * q);
                    }
                } else {                                                           // ln sigma -> bucket, edge flag
                    uint32_t packed[8];
                    uint32_t fm = 0;                                               // bit j: element j is decided by hyper_fix_kernel
#pragma unroll
                    for (int j = 0; j < 32; ++j) {
                        const float u = fminf(fmaxf(f[j], E.ln_lo), E.ln_hi);
                        f[j] = u;
                        const float t = fmaf(u - E.ln_lo, E.t_scale, 0.5f);
                        const float tf = floorf(t);
                        int k = int(tf);
                        k = k < 0 ? 0 : (k > E.n_buckets - 1 ? E.n_buckets - 1 : k);
                        const float fr = t - tf;
                        if (fminf(fr, 1.0f - fr) < xpatch * __shfl_sync(0xFFFFFFFFu, wl, j)) fm |= 1u << j;
                        if ((j & 3) == 0) packed[j >> 2] = uint32_t(k); else packed[j >> 2] |= uint32_t(k) << (8 * (j & 3));
                    }
                    if (!live) fm = 0;
                    // one atomic per warp and chunk instead of one per flagged element: 1.2 % of a million elements on a
                    // single address serialised in L2 and stretched this epilogue to 6-28 us
                    const uint32_t cnt = __popc(fm);
                    uint32_t incl = cnt;
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) {
                        const uint32_t o = __shfl_up_sync(0xFFFFFFFFu, incl, d);
                        if (lane >= d) incl += o;
                    }
                    const uint32_t total = __shfl_sync(0xFFFFFFFFu, incl, 31);
                    flush_pending();                                               // the previous chunk's slots have arrived by now
                    if (total) {
                        if (lane == 31) pend_base = atomicAdd(E.fix_count, total);
                        pend_fm = fm; pend_off = incl - cnt; pend_e0 = e0; pend_total = total;
                    }
                    if (live) {
                        st_global_256(E.idx + e0, packed);
                        if (E.lnscale) {
#pragma unroll
                            for (int q = 0; q < 4; ++q) st_global_256(E.lnscale + e0 + 8 * q, f + 8 * q);
                        }
                    }
                }
            }
            flush_pending();
        } else {
            for (int c0 = half * 32; c0 < p.BN; c0 += 64) {
                // the chunk's 32 biases are requested BEFORE the accumulator load is waited for: with ~225 KB of shared memory the L1
                // is a few KB, a bias load is an L2 round trip, and behind the TMEM wait it was a second one in a row per chunk
                float4 bb[8];
#pragma unroll
                for (int j = 0; j < 8; ++j) bb[j] = __ldg(reinterpret_cast<const float4 *>(bias + c0) + j);
                uint32_t v[32];
                tmem_ld32(t_row + uint32_t(c0), v);
                if (!inb) continue;
                const int n = tc.nt * p.BN + c0;                  // 32 consecutive packed columns, one store run
                const long long pix = ((long long)img * p.H + y) * p.W + x;
                const long long o = MODE == EPI_MU ? pix * p.E.out_stride + n : epi_offset(p.E, img, y, x, p.H, p.W, n);
                bf16 *dst = reinterpret_cast<bf16 *>(p.E.out) + o;
                float f[32];
                if (p.E.act == ACT_GELU) {
#pragma unroll
                    for (int j = 0; j < 32; j += 4) {
                        const float4 b4 = bb[j >> 2];
                        gelu_bias2(__uint_as_float(v[j]), __uint_as_float(v[j + 1]), b4.x, b4.y, f[j], f[j + 1]);
                        gelu_bias2(__uint_as_float(v[j + 2]), __uint_as_float(v[j + 3]), b4.z, b4.w, f[j + 2], f[j + 3]);
                    }
                } else {
#pragma unroll
                    for (int j = 0; j < 32; j += 4) {
                        const float4 b4 = bb[j >> 2];
                        f[j] = __uint_as_float(v[j]) + b4.x; f[j + 1] = __uint_as_float(v[j + 1]) + b4.y;
                        f[j + 2] = __uint_as_float(v[j + 2]) + b4.z; f[j + 3] = __uint_as_float(v[j + 3]) + b4.w;
                    }
                }
                if (MODE == EPI_MU) {
                    // R21: f[j] is the candidate mean mu^k of channel n + j, used where the element belongs to partition
                    // k (y = r + mu^k); elsewhere the mean used so far is carried over.  y travels as
                    // the pair (r, mu): r is an integer, exact in bf16, so only mu is rounded between the steps.
                    const EpiParams &E = p.E;
                    const uint4 *rs = reinterpret_cast<const uint4 *>(E.sym + pix * E.c_y + n);
                    const uint4 *ms = reinterpret_cast<const uint4 *>(E.y_in + pix * E.in_stride + E.c_y + n);
                    const int q = 2 * (y & 1) + (x & 1);
                    float rr[32];
#pragma unroll
                    for (int q4 = 0; q4 < 4; ++q4) {
                        const uint4 r4 = rs[q4], m4 = ms[q4];
                        const int16_t *re = reinterpret_cast<const int16_t *>(&r4);
                        const bf16 *me = reinterpret_cast<const bf16 *>(&m4);
#pragma unroll
                        for (int e = 0; e < 8; ++e) {
                            const int j = q4 * 8 + e;
                            const int part = (q + (4 * (n + j)) / E.c_y) & 3;
                            const float r = float(re[e]);
                            if (part == E.mu_step) {
                                if (E.mu_tap) E.mu_tap[pix * E.c_y + n + j] = f[j];
                                if (E.yhat_tap) E.yhat_tap[pix * E.c_y + n + j] = r + f[j];
                            } else {
                                f[j] = __bfloat162float(me[e]);                   // 0 on partitions not decoded yet
                            }
                            rr[j] = part <= E.mu_step ? r : 0.0f;
                            if (E.mu_last) f[j] += r;                             // last step: every partition is decoded
                        }
                    }
                    if (!E.mu_last) {                                             // r block, then (below) the mu block
#pragma unroll
                        for (int q4 = 0; q4 < 4; ++q4) {
                            uint4 o4;
                            __nv_bfloat162 *oe = reinterpret_cast<__nv_bfloat162 *>(&o4);
#pragma unroll
                            for (int e = 0; e < 4; ++e) oe[e] = __floats2bfloat162_rn(rr[q4 * 8 + 2 * e], rr[q4 * 8 + 2 * e + 1]);
                            reinterpret_cast<uint4 *>(dst)[q4] = o4;
                        }
                        dst += E.c_y;
                    }
                }
                if (MODE == EPI_NHWC && p.E.out_f32) {                   // fp32 output (the encoder's unquantised latent)
                    float *df = reinterpret_cast<float *>(p.E.out) + o;
#pragma unroll
                    for (int q = 0; q < 4; ++q) st_global_256(df + 8 * q, f + 8 * q);
                    continue;
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
                // A thread owns a pixel row, so every lane of a store touches its own cache line: 256-bit stores (two per 32-column
                // run instead of four of 128 bits) halve the L1 wavefronts -- the 1x1 unfold conv (A5: 2 k-blocks per 64 KB of output)
                // is bound by exactly these stores.
                uint32_t o16[16];
#pragma unroll
                for (int e = 0; e < 16; ++e) {
                    const __nv_bfloat162 h2 = __floats2bfloat162_rn(f[2 * e], f[2 * e + 1]);
                    o16[e] = *reinterpret_cast<const uint32_t *>(&h2);
                }
                if ((reinterpret_cast<uintptr_t>(dst) & 31u) == 0) {
                    st_global_256(dst, o16);
                    st_global_256(dst + 16, o16 + 8);
                } else {
#pragma unroll
                    for (int q = 0; q < 4; ++q)
                        reinterpret_cast<uint4 *>(dst)[q] = make_uint4(o16[4 * q], o16[4 * q + 1], o16[4 * q + 2], o16[4 * q + 3]);
                }
            }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) { if (pair_rank < 0) mbar_arrive(tempty0 + 8u * acc); else mbar_arrive_cluster(tempty0 + 8u * acc); }
    }
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
        for (int a = 0; a < 2; ++a) { mbar_init(tfull_bar(a), 1); mbar_init(tempty_bar(a), 8); }
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
    pdl_grid_sync();                                                 // the predecessor kernel's output is complete and visible from here on

    if (warp == 0) {
        // ===================== TMA producer =====================
        if (elect_one()) {
            int stage = 0; uint32_t phase = 0;
            for (int tile = blockIdx.x; tile < p.total_tiles; tile += gridDim.x) {
                const TileCoord tc = tile_coord(p, tile);
                const int grp = group_of(p, tc.img);
                for (int kb = 0; kb < kblocks; ++kb) {
                    const int tap = kb / p.slabs, slab = kb - tap * p.slabs;
                    const int dy = p.taps == 9 ? tap / 3 - 1 : 0, dx = p.taps == 9 ? tap % 3 - 1 : 0;
                    mbar_wait(empty_bar(stage), phase ^ 1);
                    const uint32_t a_dst = smem_base + stage * stage_bytes, b_dst = a_dst + kABytes;
                    mbar_expect_tx(full_bar(stage), stage_bytes);
                    tma_load_4d(a_dst, &tmap_a, full_bar(stage), slab * kSlabK, tc.x0 + dx, tc.y0 + dy, p.tap_img ? tc.img * p.taps + tap : tc.img);
                    tma_load_3d(b_dst, &tmap_b, full_bar(stage), slab * kSlabK, tc.nt * p.BN, grp * p.taps + tap);
                    if (++stage == kStages) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer =====================
        if (elect_one()) {
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
        epilogue_warps<MODE>(p, tmem_base, tfull_bar(0), tempty_bar(0), warp, lane);
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(tmem_cols) : "memory");
    }
}


// ---------------------------------------------------------------------------------------------------------------
// Halo variant for 3x3 convs.  The tile is 16 rows x 8 columns of pixels.  Per 64-channel slab ONE TMA box
// {64 ch, 10, 18} brings the tile plus its 1-pixel halo (zero-filled outside the image); halo pixel (hy, hx) lands at
// (hy * 10 + hx) * 128 B, 128B-swizzled relative to the 1024-aligned stage base.  Tap (dy, dx) then needs no data
// movement at all: its A operand is the same buffer viewed from start + (dy * 10 + dx) * 128 B with a stride of
// 10 * 128 = 1280 B between 8-row groups (one image row of the tile = one 8-row core-matrix group), because the
// tensor core applies the 128B swizzle to absolute shared-memory address bits.  L2->SM traffic for A drops from
// 9 x 16 KB to 22.5 KB per slab -- the first-pass kernel was bound by exactly that traffic.
// When all weight tiles of a (group, n-tile) fit the B ring (A9: 9 taps x 2 KB) they stay resident across tiles.
constexpr int kHaloTH = 16, kHaloTW = 8;
constexpr int kHaloRowPitch = (kHaloTW + 2) * 128;                            // 1280 B
constexpr int kHaloBytes = (kHaloTH + 2) * (kHaloTW + 2) * 128;              // 23040 B = one TMA box
constexpr int kHaloStage = (kHaloBytes + 1023) / 1024 * 1024;                // 23552 B
constexpr int kHaloAStages = 2;                  // an A halo stage lasts 9 k-blocks; the B ring is what must be deep

__device__ __forceinline__ uint64_t umma_desc_sw128_sbo(uint32_t saddr, uint32_t sbo_bytes)
{
    return uint64_t((saddr & 0x3FFFFu) >> 4) | (uint64_t(1) << 16) | (uint64_t(sbo_bytes >> 4) << 32) | (uint64_t(1) << 46) |
           (uint64_t(2) << 61);
}

template <int MODE, bool RESIDENT>
__global__ void __launch_bounds__(kThreads, 1)
conv_halo_kernel(const __grid_constant__ CUtensorMap tmap_a, const __grid_constant__ CUtensorMap tmap_b, const TcParams p,
                 const int nb_stages, const int na_stages)
{
    constexpr bool b_resident = RESIDENT;
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t b_bytes = uint32_t(p.BN) * 128u;                             // multiple of 2 KB
    const uint32_t b_base = smem_base + na_stages * kHaloStage;
    const uint32_t bar_base = b_base + uint32_t(nb_stages) * b_bytes;
    auto afull = [&](int s) { return bar_base + 8u * s; };
    auto aempty = [&](int s) { return bar_base + 8u * (na_stages + s); };
    const uint32_t misc = bar_base + 8u * (2 * na_stages);
    const uint32_t tfull0 = misc, tempty0 = misc + 16u, bres_full = misc + 32u, bfree = misc + 40u, tmem_slot = misc + 48u;
    const uint32_t bbar = misc + 64u;
    auto bfull = [&](int s) { return bbar + 8u * s; };
    auto bempty = [&](int s) { return bbar + 8u * (nb_stages + s); };
    volatile uint32_t *tmem_slot_ptr = reinterpret_cast<volatile uint32_t *>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int btiles = 9 * p.slabs;                                             // weight tiles per output tile
    uint32_t tmem_cols = 32;
    while (tmem_cols < uint32_t(2 * p.BN)) tmem_cols <<= 1;

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmap_a) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmap_b) : "memory");
        for (int s = 0; s < na_stages; ++s) { mbar_init(afull(s), 1); mbar_init(aempty(s), 1); }
        for (int s = 0; s < nb_stages; ++s) { mbar_init(bfull(s), 1); mbar_init(bempty(s), 1); }
        for (int a = 0; a < 2; ++a) { mbar_init(tfull0 + 8u * a, 1); mbar_init(tempty0 + 8u * a, 8); }
        mbar_init(bres_full, 1);
        mbar_init(bfree, 1);
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
    pdl_grid_sync();                                                 // the predecessor kernel's output is complete and visible from here on

    // weight-set key of a tile: resident weights are reloaded only when it changes
    auto tile_key = [&](const TileCoord &tc) { return group_of(p, tc.img) * p.n_tiles + tc.nt; };

    if (warp == 0) {
        // ===================== TMA producer =====================
        if (elect_one()) {
            int sa = 0, sb = 0; uint32_t pa = 0, pb = 0, pfree = 0;
            int prev_key = -1;
            for (int tile = blockIdx.x; tile < p.total_tiles; tile += gridDim.x) {
                const TileCoord tc = tile_coord(p, tile);
                const int grp = group_of(p, tc.img);
                if (b_resident) {
                    const int key = tile_key(tc);
                    if (key != prev_key) {
                        if (prev_key >= 0) { mbar_wait(bfree, pfree); pfree ^= 1; }     // MMAs on the old weights retired
                        mbar_expect_tx(bres_full, uint32_t(btiles) * b_bytes);
                        for (int bt = 0; bt < btiles; ++bt) {
                            const int slab = bt / 9, tap = bt - slab * 9;
                            tma_load_3d(b_base + uint32_t(bt) * b_bytes, &tmap_b, bres_full, slab * kSlabK, tc.nt * p.BN, grp * 9 + tap);
                        }
                        prev_key = key;
                    }
                }
                for (int slab = 0; slab < p.slabs; ++slab) {
                    mbar_wait(aempty(sa), pa ^ 1);
                    mbar_expect_tx(afull(sa), kHaloBytes);
                    tma_load_4d(smem_base + sa * kHaloStage, &tmap_a, afull(sa), slab * kSlabK, tc.x0 - 1, tc.y0 - 1, tc.img);
                    if (++sa == na_stages) { sa = 0; pa ^= 1; }
                    if (!b_resident) {
                        for (int tap = 0; tap < 9; ++tap) {
                            mbar_wait(bempty(sb), pb ^ 1);
                            mbar_expect_tx(bfull(sb), b_bytes);
                            tma_load_3d(b_base + uint32_t(sb) * b_bytes, &tmap_b, bfull(sb), slab * kSlabK, tc.nt * p.BN, grp * 9 + tap);
                            if (++sb == nb_stages) { sb = 0; pb ^= 1; }
                        }
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer =====================
        if (elect_one()) {
            const uint32_t idesc = umma_idesc_bf16(kTileM, p.BN);
            // descriptor halves: lo = start >> 4 | LBO(1) << 16; hi = SBO >> 4 | version 1 << 14 | SWIZZLE_128B << 29
            const uint32_t a_hi = uint32_t(kHaloRowPitch >> 4) | (1u << 14) | (2u << 29);
            const uint32_t b_hi = uint32_t(1024 >> 4) | (1u << 14) | (2u << 29);
            const uint32_t a_lo0 = ((smem_base & 0x3FFFFu) >> 4) | (1u << 16);
            const uint32_t b_lo0 = ((b_base & 0x3FFFFu) >> 4) | (1u << 16);
            const uint32_t b_step = b_bytes >> 4;
            int sa = 0, sb = 0; uint32_t pa = 0, pb = 0, pres = 0;
            int prev_key = -1;
            int it = 0;
            TileCoord tc = tile_coord(p, blockIdx.x);
            for (int tile = blockIdx.x; tile < p.total_tiles; tile += gridDim.x, ++it) {
                const int acc = it & 1;
                const uint32_t acc_phase = (it >> 1) & 1;
                if (b_resident) {
                    const int key = tile_key(tc);
                    if (key != prev_key) { mbar_wait(bres_full, pres); pres ^= 1; prev_key = key; }
                }
                mbar_wait(tempty0 + 8u * acc, acc_phase ^ 1);
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + uint32_t(acc * p.BN);
                for (int slab = 0; slab < p.slabs; ++slab) {
                    mbar_wait(afull(sa), pa);
                    tc_fence_after();
                    const uint32_t a_lo = a_lo0 + uint32_t(sa) * (kHaloStage >> 4);
                    uint32_t b_lo = b_lo0 + uint32_t(slab * 9) * b_step;                 // resident: tile (slab, tap)
#pragma unroll
                    for (int tap = 0; tap < 9; ++tap) {
                        if (!b_resident) {
                            mbar_wait(bfull(sb), pb);
                            tc_fence_after();
                            b_lo = b_lo0 + uint32_t(sb) * b_step;
                        }
                        const uint32_t a_tap = a_lo + uint32_t(((tap / 3) * (kHaloTW + 2) + tap % 3) * 128 >> 4);
#pragma unroll
                        for (int k = 0; k < kSlabK / 16; ++k)                              // 32 bytes = +2 descriptor units
                            umma_bf16_lh(d_tmem, a_tap + 2 * k, a_hi, b_lo + 2 * k, b_hi, idesc, uint32_t(slab | tap | k));
                        if (!b_resident) {
                            umma_commit(bempty(sb));
                            if (++sb == nb_stages) { sb = 0; pb ^= 1; }
                        } else {
                            b_lo += b_step;
                        }
                    }
                    umma_commit(aempty(sa));
                    if (++sa == na_stages) { sa = 0; pa ^= 1; }
                }
                umma_commit(tfull0 + 8u * acc);
                const int next = tile + gridDim.x;
                if (next < p.total_tiles) {
                    tc = tile_coord(p, next);
                    if (b_resident && tile_key(tc) != prev_key) umma_commit(bfree);      // the next tile swaps the weights
                }
            }
        }
    } else {
        epilogue_warps<MODE>(p, tmem_base, tfull0, tempty0, warp, lane);
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(tmem_cols) : "memory");
    }
}

// ---------------------------------------------------------------------------------------------------------------
// CTA-pair halo conv (cta_group::2) for the streamed-weight layers (A8).  Measured on the single-CTA kernel: the MMA
// thread spent ~60 % of its time waiting for weight stages -- four 32 KB stages buffer 1.1 us of tensor work, about one
// L2 round trip.  Here two CTAs of a cluster take two x-adjacent tiles of the same image and n-tile (same weights) and
// run ONE M = 256 MMA; each CTA stores only its half of every weight tile (BN/2 rows = 16 KB), so the same shared memory
// holds a ring twice as deep in k-blocks and every SM pulls half the weight bytes.  Leader = rank 0 issues the MMAs;
// barriers it waits on live in its shared memory (the peer's TMA and epilogue warps signal them through the cluster
// window); tcgen05.commit arrivals are multicast to both CTAs.
template <int MODE>
__global__ void __launch_bounds__(kThreads, 1)
conv_halo_pair_kernel(const __grid_constant__ CUtensorMap tmap_a, const __grid_constant__ CUtensorMap tmap_bh, const TcParams p,
                      const int nb_stages, const int na_stages)
{
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bh_bytes = uint32_t(p.BN) * 64u;                              // this CTA's half of a weight tile
    const uint32_t b_base = smem_base + na_stages * kHaloStage;
    const uint32_t bar_base = b_base + uint32_t(nb_stages) * bh_bytes;
    auto afull = [&](int s) { return bar_base + 8u * s; };
    auto aempty = [&](int s) { return bar_base + 8u * (na_stages + s); };
    const uint32_t misc = bar_base + 8u * (2 * na_stages);
    const uint32_t tfull0 = misc, tempty0 = misc + 16u, tmem_slot = misc + 48u;
    const uint32_t bbar = misc + 64u;
    auto bfull = [&](int s) { return bbar + 8u * s; };
    auto bempty = [&](int s) { return bbar + 8u * (nb_stages + s); };
    volatile uint32_t *tmem_slot_ptr = reinterpret_cast<volatile uint32_t *>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    const int pair0 = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;
    uint32_t tmem_cols = 32;
    while (tmem_cols < uint32_t(2 * p.BN)) tmem_cols <<= 1;

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmap_a) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmap_bh) : "memory");
        for (int s = 0; s < na_stages; ++s) { mbar_init(afull(s), 1); mbar_init(aempty(s), 1); }
        for (int s = 0; s < nb_stages; ++s) { mbar_init(bfull(s), 1); mbar_init(bempty(s), 1); }
        for (int a = 0; a < 2; ++a) { mbar_init(tfull0 + 8u * a, 1); mbar_init(tempty0 + 8u * a, 16); }     // 8 warps x 2 CTAs
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    cluster_sync_all();
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "r"(tmem_cols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;
    pdl_grid_sync();                                                 // the predecessor kernel's output is complete and visible from here on

    if (warp == 0) {
        // ===================== TMA producer (both CTAs): own halo tile, own half of every weight tile =====================
        if (elect_one()) {
            int sa = 0, sb = 0; uint32_t pa = 0, pb = 0;
            for (int tile = pair0; tile < p.total_tiles; tile += n_pairs) {
                const TileCoord tc = tile_coord_pair(p, tile, int(rank));          // may lie past the image: an all-zero tile
                const int grp = group_of(p, tc.img);
                for (int slab = 0; slab < p.slabs; ++slab) {
                    mbar_wait(aempty(sa), pa ^ 1);
                    if (rank == 0) mbar_expect_tx(afull(sa), 2 * kHaloBytes);
                    tma_load_4d_pair(smem_base + sa * kHaloStage, &tmap_a, mapa_rank(afull(sa), 0), slab * kSlabK, tc.x0 - 1, tc.y0 - 1, tc.img);
                    if (++sa == na_stages) { sa = 0; pa ^= 1; }
                    for (int tap = 0; tap < 9; ++tap) {
                        mbar_wait(bempty(sb), pb ^ 1);
                        if (rank == 0) mbar_expect_tx(bfull(sb), 2 * bh_bytes);
                        // transposed map: the k-block the MMA thread pairs with view (tap / 3, tap % 3) holds image tap (tap % 3, tap / 3)
                        const int wtap = p.xpose ? (tap % 3) * 3 + tap / 3 : tap;
                        tma_load_3d_pair(b_base + uint32_t(sb) * bh_bytes, &tmap_bh, mapa_rank(bfull(sb), 0), slab * kSlabK,
                                         tc.nt * p.BN + int(rank) * (p.BN >> 1), grp * 9 + wtap);
                        if (++sb == nb_stages) { sb = 0; pb ^= 1; }
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer: leader CTA only =====================
        if (rank == 0 && elect_one()) {
            const uint32_t idesc = umma_idesc_bf16(2 * kTileM, p.BN);
            const uint32_t a_hi = uint32_t(kHaloRowPitch >> 4) | (1u << 14) | (2u << 29);
            const uint32_t b_hi = uint32_t(1024 >> 4) | (1u << 14) | (2u << 29);
            const uint32_t a_lo0 = ((smem_base & 0x3FFFFu) >> 4) | (1u << 16);
            const uint32_t b_lo0 = ((b_base & 0x3FFFFu) >> 4) | (1u << 16);
            const uint32_t b_step = bh_bytes >> 4;
            int sa = 0, sb = 0; uint32_t pa = 0, pb = 0;
            int it = 0;
            for (int tile = pair0; tile < p.total_tiles; tile += n_pairs, ++it) {
                const int acc = it & 1;
                const uint32_t acc_phase = (it >> 1) & 1;
                mbar_wait_cluster(tempty0 + 8u * acc, acc_phase ^ 1);
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + uint32_t(acc * p.BN);
                for (int slab = 0; slab < p.slabs; ++slab) {
                    mbar_wait_cluster(afull(sa), pa);
                    tc_fence_after();
                    const uint32_t a_lo = a_lo0 + uint32_t(sa) * (kHaloStage >> 4);
#pragma unroll
                    for (int tap = 0; tap < 9; ++tap) {
                        mbar_wait_cluster(bfull(sb), pb);
                        tc_fence_after();
                        const uint32_t b_lo = b_lo0 + uint32_t(sb) * b_step;
                        const uint32_t a_tap = a_lo + uint32_t(((tap / 3) * (kHaloTW + 2) + tap % 3) * 128 >> 4);
#pragma unroll
                        for (int k = 0; k < kSlabK / 16; ++k)
                            umma2_bf16_lh(d_tmem, a_tap + 2 * k, a_hi, b_lo + 2 * k, b_hi, idesc, uint32_t(slab | tap | k));
                        umma2_commit_both(bempty(sb));
                        if (++sb == nb_stages) { sb = 0; pb ^= 1; }
                    }
                    umma2_commit_both(aempty(sa));
                    if (++sa == na_stages) { sa = 0; pa ^= 1; }
                }
                umma2_commit_both(tfull0 + 8u * acc);
            }
        }
    } else {
        epilogue_warps<MODE>(p, tmem_base, tfull0, mapa_rank(tempty0, 0), warp, lane, int(rank));
    }

    tc_fence_before();
    cluster_sync_all();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(tmem_cols) : "memory");
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
            std::string &err, CUtensorMapSwizzle swz = CU_TENSOR_MAP_SWIZZLE_128B)
{
    EncodeTiledFn fn = encode_fn();
    if (!fn) { err = "cuTensorMapEncodeTiled entry point not found"; return false; }
    cuuint32_t ones[5] = {1, 1, 1, 1, 1};
    CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, rank, const_cast<void *>(base), dims, strides_bytes, box, ones,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, swz, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
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

bool tc_encode_2d(CUtensorMap *tm, const void *base, unsigned long long dim0, unsigned long long dim1, unsigned box0, unsigned box1,
                  std::string &err)
{
    cuuint64_t dims[2] = {dim0, dim1};
    cuuint64_t strides[1] = {dim0 * 2};
    cuuint32_t box[2] = {box0, box1};
    return encode(tm, base, 2, dims, strides, box, err);
}

bool tc_encode_3d(CUtensorMap *tm, const void *base, unsigned long long d0, unsigned long long d1, unsigned long long d2, unsigned b0,
                  unsigned b1, unsigned b2, std::string &err)
{
    cuuint64_t dims[3] = {d0, d1, d2};
    cuuint64_t strides[2] = {d0 * 2, d0 * d1 * 2};
    cuuint32_t box[3] = {b0, b1, b2};
    return encode(tm, base, 3, dims, strides, box, err);
}

bool tc_make_weight_tmap(ConvLayer &L, std::string &err, int block_n)
{
    L.use_tc = false;
    if (L.c_in % kSlabK || L.n_pad % 16) return true;                  // not eligible: stays on the CUDA-core kernel
    L.block_n = (block_n > 0 && L.n_pad % block_n == 0) ? block_n : pick_block_n(L.n_pad);
    if (L.block_n != 16 && L.block_n % 32) return true;                // epilogue works on 32-column runs
    cuuint64_t dims[3] = {cuuint64_t(L.c_in), cuuint64_t(L.n_pad), cuuint64_t(L.groups) * L.taps};
    cuuint64_t strides[2] = {cuuint64_t(L.c_in) * 2, cuuint64_t(L.c_in) * 2 * L.n_pad};
    cuuint32_t box[3] = {cuuint32_t(kSlabK), cuuint32_t(L.block_n), 1};
    if (!encode(&L.tmap_w, L.w, 3, dims, strides, box, err)) return false;
    L.has_half_map = false;
    if (L.taps == 9 && L.block_n % 32 == 0) {                              // CTA-pair kernel: each CTA loads BN/2 rows
        cuuint32_t boxh[3] = {cuuint32_t(kSlabK), cuuint32_t(L.block_n / 2), 1};
        if (!encode(&L.tmap_w_half, L.w, 3, dims, strides, boxh, err)) return false;
        L.has_half_map = true;
    }
    L.use_tc = true;
    return true;
}

bool tc_make_act_tmap(CUtensorMap *tm, const bf16 *base, int n_img, int H, int W, int C, int tile_h, int tile_w, std::string &err,
                      bool swizzle, int pix_stride)
{
    const cuuint64_t ps = cuuint64_t(pix_stride > 0 ? pix_stride : C) * 2;      // bytes between pixels
    cuuint64_t dims[4] = {cuuint64_t(C), cuuint64_t(W), cuuint64_t(H), cuuint64_t(n_img)};
    cuuint64_t strides[3] = {ps, ps * W, ps * W * H};
    cuuint32_t box[4] = {cuuint32_t(kSlabK), cuuint32_t(tile_w), cuuint32_t(tile_h), 1};
    return encode(tm, base, 4, dims, strides, box, err, swizzle ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE);
}

bool tc_make_halo_tmap(CUtensorMap *tm, const bf16 *base, int n_img, int H, int W, int C, std::string &err)
{
    return tc_make_act_tmap(tm, base, n_img, H, W, C, kHaloTH + 2, kHaloTW + 2, err);
}

// The halo tile is 16 map rows x 8 map columns.  With the image's y as the map's dimension 1 the same tile covers 8 image rows x
// 16 image columns; whichever orientation pads the image to fewer tiles is used (A8 stage 1 at 68 x 120: 75 tiles against 72).
bool halo_prefers_transposed(int H, int W)
{
    const long normal = long((H + kHaloTH - 1) / kHaloTH) * ((W + kHaloTW - 1) / kHaloTW);
    const long xposed = long((W + kHaloTH - 1) / kHaloTH) * ((H + kHaloTW - 1) / kHaloTW);
    return xposed < normal && H > kHaloTW;             // (the pair kernel wants more than one tile width along map dimension 1)
}

// Same activation, dimensions 1 and 2 exchanged: {C, H, W, n_img} with strides {row, pixel, image}; box {64, 10 rows, 18 columns}.
bool tc_make_halo_tmap_transposed(CUtensorMap *tm, const bf16 *base, int n_img, int H, int W, int C, std::string &err)
{
    const cuuint64_t ps = cuuint64_t(C) * 2;
    cuuint64_t dims[4] = {cuuint64_t(C), cuuint64_t(H), cuuint64_t(W), cuuint64_t(n_img)};
    cuuint64_t strides[3] = {ps * W, ps, ps * W * H};
    cuuint32_t box[4] = {cuuint32_t(kSlabK), cuuint32_t(kHaloTW + 2), cuuint32_t(kHaloTH + 2), 1};
    return encode(tm, base, 4, dims, strides, box, err);
}

cudaError_t configure_conv_tc_kernels()
{
    cudaError_t e = cudaSuccess;
    auto set = [&](auto kern) { if (e == cudaSuccess) e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024); };
    set(conv_halo_pair_kernel<EPI_PS2>); set(conv_halo_pair_kernel<EPI_HEAD>); set(conv_halo_pair_kernel<EPI_MU>);
    set(conv_halo_kernel<EPI_NHWC, true>); set(conv_halo_kernel<EPI_NHWC, false>);
    set(conv_halo_kernel<EPI_PS2, true>); set(conv_halo_kernel<EPI_PS2, false>);
    set(conv_halo_kernel<EPI_HEAD, false>);
    set(conv_halo_kernel<EPI_MU, true>); set(conv_halo_kernel<EPI_MU, false>);
    set(conv_halo_kernel<EPI_FINAL, true>); set(conv_halo_kernel<EPI_FINAL, false>);
    set(conv_tc_kernel<EPI_NHWC>); set(conv_tc_kernel<EPI_PS2>); set(conv_tc_kernel<EPI_HEAD>); set(conv_tc_kernel<EPI_MU>);
    set(conv_tc_kernel<EPI_FINAL>);
    return e;
}

cudaError_t launch_conv_halo_pair(const ConvLayer &L, const ConvProblem &P, const CUtensorMap &tmap_halo, const EpiParams &E, int num_sms,
                                  LaunchStream st, bool transposed)
{
    if (L.taps != 9 || !L.has_half_map || (E.mode != EPI_PS2 && E.mode != EPI_HEAD && E.mode != EPI_MU)) return cudaErrorInvalidValue;
    TcParams p{};
    p.H = P.H; p.W = P.W;
    p.xpose = transposed ? 1 : 0;
    p.reverse = P.reverse ? 1 : 0;
    p.n_img_m = P.n_img; p.Hm = transposed ? P.W : P.H; p.Wm = transposed ? P.H : P.W;
    p.TH = kHaloTH; p.TW = kHaloTW;
    p.flat = 0; p.tw_shift = 3;
    p.tiles_y = (p.Hm + kHaloTH - 1) / kHaloTH;
    p.tiles_x = (p.Wm + kHaloTW - 1) / kHaloTW;
    p.tiles_img = p.tiles_y * p.tiles_x;
    const int pairs = (p.tiles_img + 1) / 2;                       // schedule unit = (image, pair of consecutive tiles, n tile)
    p.taps = 9; p.slabs = L.c_in / kSlabK;
    p.BN = L.block_n; p.n_tiles = L.n_pad / L.block_n; p.n_real = L.n; p.n_pad = L.n_pad;
    p.groups = L.groups;
    p.total_tiles = p.n_img_m * pairs * p.n_tiles;
    p.fd_ntiles = make_fastdiv(p.n_tiles); p.fd_tx = make_fastdiv(p.tiles_x); p.fd_ty = make_fastdiv(p.tiles_y);
    p.fd_pairs = make_fastdiv(pairs);
    p.fd_groups = make_fastdiv(p.groups);
    p.bias = L.bias;
    p.E = E;
    const size_t bh_bytes = size_t(L.block_n) * 64;
    const int na = kHaloAStages;
    int nb = int((227 * 1024 - 1024 - size_t(na) * kHaloStage - 2048) / bh_bytes);
    if (nb > 12) nb = 12;
    if (nb < 2) return cudaErrorInvalidValue;
    const size_t smem = 1024 + size_t(na) * kHaloStage + size_t(nb) * bh_bytes + 256 + 16 * size_t(nb) + 16 * size_t(na);
    const int clusters = p.total_tiles < num_sms / 2 ? p.total_tiles : num_sms / 2;
    if (E.mode == EPI_HEAD) return launch_pdl(conv_halo_pair_kernel<EPI_HEAD>, 2 * clusters, kThreads, smem, st, 2, tmap_halo, L.tmap_w_half, p, nb, na);
    if (E.mode == EPI_MU) return launch_pdl(conv_halo_pair_kernel<EPI_MU>, 2 * clusters, kThreads, smem, st, 2, tmap_halo, L.tmap_w_half, p, nb, na);
    return launch_pdl(conv_halo_pair_kernel<EPI_PS2>, 2 * clusters, kThreads, smem, st, 2, tmap_halo, L.tmap_w_half, p, nb, na);
}

cudaError_t launch_conv_halo(const ConvLayer &L, const ConvProblem &P, const CUtensorMap &tmap_halo, const EpiParams &E, int num_sms,
                             LaunchStream st)
{
    if (L.taps != 9) return cudaErrorInvalidValue;
    TcParams p{};
    p.H = P.H; p.W = P.W;
    p.n_img_m = P.n_img; p.Hm = P.H; p.Wm = P.W;
    p.TH = kHaloTH; p.TW = kHaloTW;
    p.flat = 0; p.tw_shift = 3;
    p.tiles_y = (P.H + kHaloTH - 1) / kHaloTH;
    p.tiles_x = (P.W + kHaloTW - 1) / kHaloTW;
    p.taps = 9; p.slabs = L.c_in / kSlabK;
    p.BN = L.block_n; p.n_tiles = L.n_pad / L.block_n; p.n_real = L.n; p.n_pad = L.n_pad;
    p.groups = L.groups;
    p.total_tiles = p.n_img_m * p.tiles_y * p.tiles_x * p.n_tiles;
    p.fd_ntiles = make_fastdiv(p.n_tiles); p.fd_tx = make_fastdiv(p.tiles_x); p.fd_ty = make_fastdiv(p.tiles_y);
    p.fd_groups = make_fastdiv(p.groups);
    p.bias = L.bias;
    p.E = E;
    const size_t b_bytes = size_t(L.block_n) * 128;
    int na = kHaloAStages;
    const size_t budget = 227 * 1024 - 1024 - size_t(na) * kHaloStage - 1024;
    const int btiles = 9 * p.slabs;
    int nb = int(budget / b_bytes);
    const int resident = btiles <= nb ? 1 : 0;
    if (resident) nb = btiles; else if (nb > 8) nb = 8;
    if (nb < 2) return cudaErrorInvalidValue;
    // small resident weights (A9) leave room: deepen the A ring so more halo loads are in flight per SM
    while (na < 8 && 1024 + size_t(na + 1) * kHaloStage + size_t(nb) * b_bytes + 2048 <= 227 * 1024) ++na;
    const size_t smem = 1024 + size_t(na) * kHaloStage + size_t(nb) * b_bytes + 256 + 16 * size_t(nb) + 16 * size_t(na);
    const int grid = p.total_tiles < num_sms ? p.total_tiles : num_sms;
    auto launch = [&](auto kern) -> cudaError_t { return launch_pdl(kern, grid, kThreads, smem, st, 1, tmap_halo, L.tmap_w, p, nb, na); };
    switch (E.mode) {
        case EPI_NHWC: return resident ? launch(conv_halo_kernel<EPI_NHWC, true>) : launch(conv_halo_kernel<EPI_NHWC, false>);
        case EPI_PS2: return resident ? launch(conv_halo_kernel<EPI_PS2, true>) : launch(conv_halo_kernel<EPI_PS2, false>);
        case EPI_HEAD: return resident ? cudaErrorInvalidValue : launch(conv_halo_kernel<EPI_HEAD, false>);
        case EPI_MU: return resident ? launch(conv_halo_kernel<EPI_MU, true>) : launch(conv_halo_kernel<EPI_MU, false>);
        default: return resident ? launch(conv_halo_kernel<EPI_FINAL, true>) : launch(conv_halo_kernel<EPI_FINAL, false>);
    }
}

cudaError_t launch_conv_tc(const ConvLayer &L, const ConvProblem &P, const CUtensorMap &tmap_in, int tile_h, int tile_w, bool flat,
                           const EpiParams &E, int num_sms, LaunchStream st)
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
    p.flat = flat ? 1 : 0;
    for (p.tw_shift = 0; (1 << p.tw_shift) < tile_w; ++p.tw_shift) {}
    p.tiles_y = (p.Hm + tile_h - 1) / tile_h;
    p.tiles_x = (p.Wm + tile_w - 1) / tile_w;
    p.taps = L.taps; p.slabs = L.c_in / kSlabK;
    p.tap_img = P.taps_are_images ? 1 : 0;
    if (p.tap_img && flat) return cudaErrorInvalidValue;
    p.BN = L.block_n; p.n_tiles = L.n_pad / L.block_n; p.n_real = L.n; p.n_pad = L.n_pad;
    p.groups = L.groups;
    p.total_tiles = p.n_img_m * p.tiles_y * p.tiles_x * p.n_tiles;
    p.fd_ntiles = make_fastdiv(p.n_tiles); p.fd_tx = make_fastdiv(p.tiles_x); p.fd_ty = make_fastdiv(p.tiles_y);
    p.fd_groups = make_fastdiv(p.groups);
    p.bias = L.bias;
    p.E = E;
    const size_t smem = size_t(kStages) * (kABytes + size_t(L.block_n) * 128) + 1024 + 256;
    const int grid = p.total_tiles < num_sms ? p.total_tiles : num_sms;
    auto launch = [&](auto kern) -> cudaError_t { return launch_pdl(kern, grid, kThreads, smem, st, 1, tmap_in, L.tmap_w, p); };
    switch (E.mode) {
        case EPI_NHWC: return launch(conv_tc_kernel<EPI_NHWC>);
        case EPI_PS2: return launch(conv_tc_kernel<EPI_PS2>);
        case EPI_HEAD: return launch(conv_tc_kernel<EPI_HEAD>);
        case EPI_MU: return launch(conv_tc_kernel<EPI_MU>);
        default: return launch(conv_tc_kernel<EPI_FINAL>);
    }
}

}  // namespace ufnvc
