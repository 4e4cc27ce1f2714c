// A7: the trunk DC block's MLP as ONE tcgen05 kernel ("DC block"):
//
//     out = x + W2 * GELU(W1 * d + b1) + b2,      d = depthwise(x) [A6],  256 -> 1024 -> 256, per pixel
//
// Unfused, the 1024-wide hidden tensor makes a 268 MB HBM round trip per block and the block is bandwidth-bound
// (DESIGN.md section 6).  Here a CTA owns 128 pixels and walks the hidden dimension in chunks of 128 columns:
//
//   GEMM1(c): Hacc[c&1] (TMEM, 128 x 128 fp32)  = d_tile (smem, 128 x 256)  x  W1[c]^T   (4 slabs x 4 UMMAs, N = 128)
//   epi(c):   Hacc -> registers -> +b1 -> GELU -> bf16 -> Hs[c&1] (smem, written directly in the K-major SWIZZLE_128B
//             layout tcgen05.mma reads; fence.proxy.async hands it to the tensor core)
//   GEMM2(c): Oacc (TMEM, 128 x 256 fp32)      += Hs[c&1] (128 x 128)  x  W2[:, c]^T     (2 slabs x 4 UMMAs, N = 256)
//
// The MMA warp issues GEMM1(c+1) before GEMM2(c), so the tensor core always has a GEMM to run while the epilogue warps
// do the GELU of chunk c.  TMEM: 256 (Oacc) + 2 x 128 (Hacc) = all 512 columns.  Shared memory: d tile 64 KB, Hs
// 2 x 32 KB, weight ring 3 x 32 KB (W1 and W2 chunks stream through it in the order the MMA warp consumes them).
// warp 0 = TMA producer, warp 1 = MMA issuer + TMEM allocator, warps 2..9 = epilogue.  Persistent, grid = #SMs.
#include <cuda.h>

#include <algorithm>
#include <cstring>

#include "epilogue.cuh"
#include "tc_ptx.cuh"
#include "ufnvc_internal.h"

namespace ufnvc {

namespace {

constexpr int kC = 256;                  // trunk width: K of GEMM1, N of GEMM2
constexpr int kHC = 128;                 // hidden columns per chunk
constexpr int kTM = 128;                 // pixels per tile
constexpr int kTrunkThreads = 320;       // single-CTA kernel: TMA warp, MMA warp, 8 epilogue warps
constexpr int kPairThreads = 512;        // CTA-pair kernel: weight TMA warp, MMA warp, 4 GELU warps, 8 drain warps, relay warp, input-tile TMA warp
static_assert(kPairThreads / 32 - 8 == int(kTrunkTileSignals), "one tile_done increment per drain warp (warps 6..13)");
constexpr int kWStages = 3;
constexpr uint32_t kSlab = 16384;        // 128 rows x 128 B
constexpr uint32_t kWStage = 32768;
constexpr uint32_t kOffA = 0, kOffHs = 4 * kSlab, kOffW = kOffHs + 4 * kSlab, kOffBar = kOffW + kWStages * kWStage;
constexpr uint32_t kTrunkSmem = kOffBar + 256 + 1024;        // + alignment slack

constexpr int kMaxHidden = 1024;         // biases travel in the kernel parameters (constant bank): warp-uniform reads
struct TrunkParams {
    int n_tiles, n_chunks, n_px;
    const float *b1, *b2;                // [hidden], [256] (device copies: the single-CTA kernel reads these)
    float hb1v[kMaxHidden];              // b1 / 2 by value (CTA-pair kernel: constant bank, warp-uniform reads)
    float b2v[kC];                       // b2 by value
    const bf16 *x;                       // residual input  [n_px][256]
    bf16 *out;                           // [n_px][256] (may alias x: a tile reads its own rows before writing them)
    uint32_t *tile_done;                 // optional: [n_tiles] counters, +1 per epilogue warp (8 per tile) once its rows are written
};

// barrier slots (8 bytes each) from kOffBar
enum : uint32_t {
    B_AFULL = 0, B_AEMPTY = 1, B_WFULL = 2, B_WEMPTY = 5, B_HACC_FULL = 8, B_HACC_EMPTY = 10, B_HS_FULL = 12, B_HS_EMPTY = 14,
    B_OFULL = 16, B_OEMPTY = 17, B_TMEM_SLOT = 18
};

}  // namespace

namespace {

__device__ __forceinline__ void st_shared_v4(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d)
{
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi)
{
    const __nv_bfloat162 h = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<const uint32_t *>(&h);
}

__global__ void __launch_bounds__(kTrunkThreads, 1)
trunk_mlp_kernel(const __grid_constant__ CUtensorMap tm_d, const __grid_constant__ CUtensorMap tm_w1,
                 const __grid_constant__ CUtensorMap tm_w2, const TrunkParams p)
{
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    auto bar = [&](uint32_t slot) { return base + kOffBar + 8u * slot; };
    volatile uint32_t *tmem_slot_ptr =
        reinterpret_cast<volatile uint32_t *>(smem_raw + (bar(B_TMEM_SLOT) - smem_u32(smem_raw)));
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int NC = p.n_chunks;

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_d) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_w1) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_w2) : "memory");
        mbar_init(bar(B_AFULL), 1); mbar_init(bar(B_AEMPTY), 1);
        for (int s = 0; s < kWStages; ++s) { mbar_init(bar(B_WFULL + s), 1); mbar_init(bar(B_WEMPTY + s), 1); }
        for (int b = 0; b < 2; ++b) {
            mbar_init(bar(B_HACC_FULL + b), 1); mbar_init(bar(B_HACC_EMPTY + b), 8);
            mbar_init(bar(B_HS_FULL + b), 8);   mbar_init(bar(B_HS_EMPTY + b), 1);
        }
        mbar_init(bar(B_OFULL), 1); mbar_init(bar(B_OEMPTY), 8);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(bar(B_TMEM_SLOT)), "r"(512u) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;
    pdl_grid_sync();                                                 // the predecessor kernel's output is complete and visible from here on

    if (warp == 0) {
        // ===================== TMA producer: d tile, then W1 / W2 chunks in MMA consumption order =====================
        if (elect_one()) {
            int ws = 0; uint32_t wp = 0, ap = 0;
            auto w_slot = [&]() {                                  // claim the next ring stage; returns its smem address
                mbar_wait(bar(B_WEMPTY + ws), wp ^ 1);
                mbar_expect_tx(bar(B_WFULL + ws), kWStage);
                return base + kOffW + uint32_t(ws) * kWStage;
            };
            auto w_next = [&]() { if (++ws == kWStages) { ws = 0; wp ^= 1; } };
            auto load_w1 = [&](int c) {                            // rows c*128.. of W1, k slabs (2st, 2st+1) per stage
                for (int st = 0; st < 2; ++st) {
                    const uint32_t dst = w_slot();
                    tma_load_2d(dst, &tm_w1, bar(B_WFULL + ws), (2 * st) * 64, c * kHC);
                    tma_load_2d(dst + kSlab, &tm_w1, bar(B_WFULL + ws), (2 * st + 1) * 64, c * kHC);
                    w_next();
                }
            };
            auto load_w2 = [&](int c) {                            // all 256 rows of W2, k slab c*128 + st*64 per stage
                for (int st = 0; st < 2; ++st) {
                    const uint32_t dst = w_slot();
                    tma_load_2d(dst, &tm_w2, bar(B_WFULL + ws), c * kHC + st * 64, 0);
                    w_next();
                }
            };
            for (int tile = blockIdx.x; tile < p.n_tiles; tile += gridDim.x) {
                mbar_wait(bar(B_AEMPTY), ap ^ 1);
                mbar_expect_tx(bar(B_AFULL), 4 * kSlab);
                for (int s = 0; s < 4; ++s) tma_load_2d(base + kOffA + s * kSlab, &tm_d, bar(B_AFULL), s * 64, tile * kTM);
                ap ^= 1;
                load_w1(0);
                if (NC > 1) load_w1(1);
                for (int c = 0; c < NC; ++c) {                     // the order the MMA warp consumes them in
                    if (c + 2 < NC) load_w1(c + 2);
                    load_w2(c);
                }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer =====================
        if (elect_one()) {
            const uint32_t idesc1 = umma_idesc_bf16(kTM, kHC), idesc2 = umma_idesc_bf16(kTM, kC);
            const uint32_t hi = uint32_t(1024 >> 4) | (1u << 14) | (2u << 29);
            auto lo = [](uint32_t addr) { return ((addr & 0x3FFFFu) >> 4) | (1u << 16); };
            const uint32_t a_lo = lo(base + kOffA), hs_lo = lo(base + kOffHs), w_lo = lo(base + kOffW);
            const uint32_t o_acc = tmem_base, h_acc = tmem_base + kC;
            int ws = 0; uint32_t wp = 0;
            uint32_t ph_hacc = 0, ph_hs = 0;                      // bit b = parity of the use count of buffer b
            auto w_wait = [&]() {
                mbar_wait(bar(B_WFULL + ws), wp);
                tc_fence_after();
                return w_lo + uint32_t(ws) * (kWStage >> 4);
            };
            auto w_release = [&]() { umma_commit(bar(B_WEMPTY + ws)); if (++ws == kWStages) { ws = 0; wp ^= 1; } };
            auto gemm1 = [&](int c) {
                const int b = c & 1;
                mbar_wait(bar(B_HACC_EMPTY + b), ((ph_hacc >> b) & 1) ^ 1);
                ph_hacc ^= 1u << b;
                tc_fence_after();
                const uint32_t d = h_acc + uint32_t(b) * kHC;
#pragma unroll
                for (int st = 0; st < 2; ++st) {
                    const uint32_t w = w_wait();
#pragma unroll
                    for (int j = 0; j < 2; ++j)
#pragma unroll
                        for (int k = 0; k < 4; ++k)
                            umma_bf16_lh(d, a_lo + uint32_t(2 * st + j) * (kSlab >> 4) + 2 * k, hi, w + uint32_t(j) * (kSlab >> 4) + 2 * k, hi,
                                         idesc1, uint32_t(st | j | k));
                    w_release();
                }
                umma_commit(bar(B_HACC_FULL + b));
            };
            int it = 0;
            for (int tile = blockIdx.x; tile < p.n_tiles; tile += gridDim.x, ++it) {
                mbar_wait(bar(B_AFULL), it & 1);
                tc_fence_after();
                // GEMM1 runs two chunks ahead of GEMM2: the epilogue frees Hacc[c&1] as soon as chunk c sits in its registers,
                // so GEMM1(c+2) is queued behind GEMM1(c+1) while the GELU of chunk c is still being computed
                gemm1(0);
                if (NC > 1) gemm1(1);
                if (NC <= 2) umma_commit(bar(B_AEMPTY));
                for (int c = 0; c < NC; ++c) {
                    if (c + 2 < NC) {
                        gemm1(c + 2);
                        if (c + 3 == NC) umma_commit(bar(B_AEMPTY));      // every GEMM1 of this tile has been issued
                    }
                    const int b = c & 1;
                    mbar_wait(bar(B_HS_FULL + b), (ph_hs >> b) & 1);
                    ph_hs ^= 1u << b;
                    if (c == 0) mbar_wait(bar(B_OEMPTY), (it & 1) ^ 1);  // previous tile's output has left TMEM
                    tc_fence_after();
#pragma unroll
                    for (int st = 0; st < 2; ++st) {
                        const uint32_t w = w_wait();
#pragma unroll
                        for (int k = 0; k < 4; ++k)
                            umma_bf16_lh(o_acc, hs_lo + uint32_t(2 * b + st) * (kSlab >> 4) + 2 * k, hi, w + 2 * k, hi, idesc2,
                                         uint32_t(c | st | k));
                        w_release();
                    }
                    umma_commit(bar(B_HS_EMPTY + b));
                }
                umma_commit(bar(B_OFULL));
            }
        }
    } else {
        // ===================== epilogue warps =====================
        const int quad = warp & 3, half = (warp - 2) >> 2;
        const int r = quad * 32 + lane;                                   // row of the tile = TMEM lane
        const uint32_t t_lane = tmem_base + (uint32_t(quad * 32) << 16);
        uint32_t ph_use = 0;
        float2 bnext = __ldg(reinterpret_cast<const float2 *>(p.b1 + half * 64) + lane);          // chunk 0
        float b2r[4];                                                     // b2[half*128 + 32 i + lane]
#pragma unroll
        for (int i = 0; i < 4; ++i) b2r[i] = __ldg(p.b2 + half * 128 + 32 * i + lane);
        int it = 0;
        for (int tile = blockIdx.x; tile < p.n_tiles; tile += gridDim.x, ++it) {
            for (int c = 0; c < NC; ++c) {
                const int b = c & 1;
                mbar_wait(bar(B_HACC_FULL + b), (ph_use >> b) & 1);
                mbar_wait(bar(B_HS_EMPTY + b), ((ph_use >> b) & 1) ^ 1);
                ph_use ^= 1u << b;
                tc_fence_after();
                // this chunk's 64 biases live 2 per lane (fetched one chunk ahead: with ~225 KB of shared memory the L1 is a few
                // KB, so a bias load in the dependent chain costs an L2 round trip); the next chunk's are requested now
                const float2 bcur = bnext;
                {
                    const int cn = c + 1 < NC ? c + 1 : 0;
                    bnext = __ldg(reinterpret_cast<const float2 *>(p.b1 + cn * kHC + half * 64) + lane);
                }
                const uint32_t hs_row = base + kOffHs + uint32_t(2 * b + half) * kSlab + uint32_t(r) * 128u;
                // both 32-column loads are in flight before the single wait: a TMEM load costs ~400 cycles while the tensor
                // core is accumulating, and it sits on the GEMM1 -> GELU -> GEMM2 critical chain
                uint32_t vv[2][32];
                tmem_ld32_nowait(t_lane + kC + uint32_t(b) * kHC + uint32_t(half * 64), vv[0]);
                tmem_ld32_nowait(t_lane + kC + uint32_t(b) * kHC + uint32_t(half * 64 + 32), vv[1]);
                tmem_ld_wait();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(B_HACC_EMPTY + b));        // chunk c is in registers: Hacc[b] may be overwritten
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                    uint32_t (&v)[32] = vv[q];
                    uint32_t pk[16];
#pragma unroll
                    for (int j = 0; j < 32; j += 2) {                     // columns q*32 + j, j+1 <- lane (q*32 + j) / 2
                        const float bx = __shfl_sync(0xFFFFFFFFu, bcur.x, q * 16 + j / 2);
                        const float by = __shfl_sync(0xFFFFFFFFu, bcur.y, q * 16 + j / 2);
                        float f0, f1;
                        gelu_bias2(__uint_as_float(v[j]), __uint_as_float(v[j + 1]), bx, by, f0, f1);
                        pk[j / 2] = pack_bf16x2(f0, f1);
                    }
#pragma unroll
                    for (int jj = 0; jj < 4; ++jj) {                      // 16-byte chunk q*4+jj of the row, 128B-swizzled
                        const uint32_t chunk = uint32_t(q * 4 + jj) ^ uint32_t(r & 7);
                        st_shared_v4(hs_row + (chunk << 4), pk[4 * jj], pk[4 * jj + 1], pk[4 * jj + 2], pk[4 * jj + 3]);
                    }
                }
                tc_fence_before();
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(B_HS_FULL + b));
            }
            // ---- output: Oacc + b2 + x -> bf16.  The residual row segment (128 columns = 16 x 16 B) is fetched BEFORE the
            // wait for the last GEMM2s, so its latency hides behind them: Oacc is single-buffered, which puts this
            // epilogue on the tile's critical path (fetched after the wait it cost ~60 % of the kernel).
            const long long row = (long long)tile * kTM + r;
            const bool inb = row < p.n_px;
            uint4 res[16];
            {
                const uint4 *rs = reinterpret_cast<const uint4 *>(p.x + row * kC + half * 128);
#pragma unroll
                for (int g = 0; g < 16; ++g) res[g] = inb ? rs[g] : make_uint4(0, 0, 0, 0);
            }
            mbar_wait(bar(B_OFULL), it & 1);
            tc_fence_after();
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                uint32_t v[32];
                const int c0 = half * 128 + q * 32;
                tmem_ld32(t_lane + uint32_t(c0), v);
                uint4 *dst = reinterpret_cast<uint4 *>(p.out + row * kC + c0);
#pragma unroll
                for (int g = 0; g < 4; ++g) {
                    const __nv_bfloat162 *re = reinterpret_cast<const __nv_bfloat162 *>(&res[q * 4 + g]);
                    float bs[8];
#pragma unroll
                    for (int e = 0; e < 8; ++e) bs[e] = __shfl_sync(0xFFFFFFFFu, b2r[q], g * 8 + e);
                    uint4 o4;
                    uint32_t *oe = reinterpret_cast<uint32_t *>(&o4);
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const float2 xr = __bfloat1622float2(re[e]);
                        oe[e] = pack_bf16x2(__uint_as_float(v[g * 8 + 2 * e]) + bs[2 * e] + xr.x,
                                            __uint_as_float(v[g * 8 + 2 * e + 1]) + bs[2 * e + 1] + xr.y);
                    }
                    if (inb) dst[g] = o4;                                 // (shuffles above need every lane)
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(B_OEMPTY));
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

namespace {

// ---------------------------------------------------------------------------------------------------------------
// CTA-pair version (cta_group::2).  The single-CTA kernel above is bound by the weight ring: every 128-pixel tile pulls
// the whole 1 MB of W1 + W2 through 96 KB of shared memory, and with ~1.5-2 us of L2 latency that ring cannot deliver
// the 122 GB/s per SM the tensor core would consume (measured: tensor pipe 42 % active, L2 throughput 21 %).  A pair of
// CTAs on one TPC runs ONE M = 256 MMA over both d tiles; each CTA stores only HALF of every weight tile (N/2 rows), so
// the bytes per SM and per tile drop to 512 KB and a ring stage now lasts a whole GEMM1 or GEMM2 chunk (1024 tensor
// cycles).  The pair's leader CTA (even cluster rank) issues all MMAs; both CTAs run their own producers and epilogue warps.
// Barriers the MMA thread waits on live in the leader (the peer signals them through the cluster window); barriers signalled
// by tcgen05.commit are multicast to both CTAs.  Warps of a CTA: 0 weight producer, 1 MMA issuer + TMEM allocator, 2..5 GELU
// (one per TMEM lane quadrant = scheduler), 6..13 output drain (two per quadrant), 14 relay and 15 input-tile producer (see
// the cluster-of-two-pairs note in the kernel).
// TMH = true: the GELU'd hidden chunk goes back into TMEM (bf16, over the fp32 columns it came from) and GEMM2 reads its
// A operand from there: no 64 KB Hs buffer (the weight ring grows from 3 to 5 stages), and per tile 256 KB of st.shared
// plus 256 KB of A-operand reads leave the shared-memory port, which TMA writes + MMA operand reads had saturated.
// (acc0, acc1) + bias -> GELU of each, returned as one bf16x2 word (low half = element 0): the form GEMM2 reads from TMEM.
// hb = (b0 / 2, b1 / 2).  With w = v / 2:  GELU(v) = w + w tanh(w (2a + 8b w^2)),  (a, b) = (0.80015708, 0.03470089) fitted to
// the erf form (max |error| 2.7e-4, rms 1.3e-4 -- a quarter of the bf16 rounding of the stored result; the three-coefficient fit
// of epilogue.cuh is 10x closer but needs a clamp and two more operations).  Five packed-fp32 operations, two MUFU.TANH and
// one pack per PAIR.  Why this form: at the tensor pipe's full rate a scheduler has 16 issue slots per 32 hidden elements, and
// clock64 around the phases of the epilogue warps showed the previous GELU (7 packed operations, 2 FMNMX, 2 MUFU, 2 bias
// shuffles, 1 pack = 14 slots per pair and 14 FMA-pipe cycles) taking 1650 of a chunk's 2048 tensor cycles on every scheduler;
// with the output drain on the same warps the hidden chunk came back too late for GEMM2 and the tensor pipe idled 45 % of
// the time.  An f16x2 version was no better (B200 issues fma.f16x2 at the same 2 cycles as fma.f32x2, and tanh.approx.f16x2
// is two MUFU operations); the floor that remains is the MUFU pipe: 4 lanes per clock = 1024 cycles per chunk.
__device__ __forceinline__ uint32_t gelu_bias2_pk(float acc0, float acc1, float hb0, float hb1)
{
    const uint64_t w = f2_fma(f2_pack(acc0, acc1), f2_pack(0.5f, 0.5f), f2_pack(hb0, hb1));
    const uint64_t pl = f2_fma(f2_pack(8.0f * 0.03470089f, 8.0f * 0.03470089f), f2_mul(w, w), f2_pack(2.0f * 0.80015708f, 2.0f * 0.80015708f));
    float u0, u1, t0, t1, g0, g1;
    f2_unpack(f2_mul(w, pl), u0, u1);
    asm("tanh.approx.f32 %0, %1;" : "=f"(t0) : "f"(u0));
    asm("tanh.approx.f32 %0, %1;" : "=f"(t1) : "f"(u1));
    f2_unpack(f2_fma(w, f2_pack(t0, t1), w), g0, g1);
    return pack_bf16x2(g0, g1);
}
__device__ __forceinline__ void ld_global_256(const void *p, uint32_t (&u)[8])
{
    asm volatile("ld.global.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];" : "=r"(u[0]), "=r"(u[1]), "=r"(u[2]), "=r"(u[3]), "=r"(u[4]), "=r"(u[5]),
                 "=r"(u[6]), "=r"(u[7]) : "l"(p));
}

constexpr bool TMH = true;     // (the shared-memory-hidden variant, TMH = false, lost the A/B and is no longer instantiated)
__global__ void __launch_bounds__(kPairThreads, 1)
trunk_mlp_pair_kernel(const __grid_constant__ CUtensorMap tm_d, const __grid_constant__ CUtensorMap tm_w1h,
                      const __grid_constant__ CUtensorMap tm_w2h, const __grid_constant__ TrunkParams p)
{
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    constexpr int NS = TMH ? 5 : 3;                            // weight-ring stages
    constexpr uint32_t offW = TMH ? kOffHs : kOffW, offBar = offW + NS * kWStage;
    // HS_FULL: one barrier per Hacc buffer and 32-column sub-step of a chunk (2 x 4)
    constexpr uint32_t B_WFULL = 2, B_WEMPTY = B_WFULL + NS, B_HACC_FULL = B_WEMPTY + NS, B_HS_FULL = B_HACC_FULL + 2,
                       B_OFULL = B_HS_FULL + 8, B_OEMPTY = B_OFULL + 1, B_PFULL = B_OEMPTY + 1, B_TMEM_SLOT = B_PFULL + NS;   // (shadow the file-scope slots)
    auto bar = [&](uint32_t slot) { return base + offBar + 8u * slot; };
    volatile uint32_t *tmem_slot_ptr =
        reinterpret_cast<volatile uint32_t *>(smem_raw + (bar(B_TMEM_SLOT) - smem_u32(smem_raw)));
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // Cluster = one CTA pair, or (preferred cluster dimension, where the GPC has room) TWO pairs that share every weight tile: each
    // of the four CTAs then fetches a quarter of it and multicasts it to its counterpart in the other pair, which halves the
    // L2 -> SM weight traffic -- the kernel moves 704 KB per CTA and tile pair, and at the tensor pipe's rate that is the whole
    // chip's L2 output bandwidth.  The pairs of a cluster walk the weight ring in lockstep; a pair that has run out
    // of tiles computes a padding tile (rows past n_px: zero-filled loads, masked stores).
    const uint32_t rank = cluster_ctarank(), nranks = cluster_nctarank();
    const uint32_t hb = rank & 1u, leader = rank & ~1u, pc = rank >> 1;      // half of the pair, the pair's MMA-issuing CTA, pair in cluster
    const bool quad = nranks == 4;
    const uint32_t pair_mask = 3u << (2 * pc), all_mask = quad ? 0xFu : 0x3u;
    const int NC = p.n_chunks;
    const int n_pairs = gridDim.x >> 1, pair0 = blockIdx.x >> 1;
    const int n_ptiles = (p.n_tiles + 1) >> 1;                       // tile pairs; a missing odd tile is all padding
    const int first_pair = pair0 - int(pc);                          // the cluster's first pair has the most tiles: its count is everyone's
    const int rounds = first_pair < n_ptiles ? (n_ptiles - first_pair + n_pairs - 1) / n_pairs : 0;

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_d) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_w1h) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_w2h) : "memory");
        mbar_init(bar(B_AFULL), 1); mbar_init(bar(B_AEMPTY), 1);
        for (int s = 0; s < NS; ++s) { mbar_init(bar(B_WFULL + s), 1); mbar_init(bar(B_WEMPTY + s), quad ? 2 : 1); mbar_init(bar(B_PFULL + s), 2); }
        for (int b = 0; b < 2; ++b) {
            mbar_init(bar(B_HACC_FULL + b), 1);
            for (int q = 0; q < 4; ++q) mbar_init(bar(B_HS_FULL + 4 * b + q), 8);         // 4 GELU warps x 2 CTAs per sub-step
        }
        mbar_init(bar(B_OFULL), 1); mbar_init(bar(B_OEMPTY), 16);                         // 8 drain warps x 2 CTAs
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    cluster_sync_all();                                              // peer barriers are initialised before anyone signals
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(bar(B_TMEM_SLOT)), "r"(512u) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;
    pdl_grid_sync();                                                 // the predecessor kernel's output is complete and visible from here on

    if (warp == 0) {
        // ===================== weight producer (both CTAs): own half of every weight tile (a quarter, multicast, in two-pair clusters) ====
        if (elect_one()) {
            const uint32_t mc_mask = (1u << rank) | (1u << (rank ^ 2u));   // this CTA and its counterpart in the other pair
            int ws = 0; uint32_t wp = 0;
            auto w_slot = [&](uint32_t &full_l) {
                mbar_wait_cluster(bar(B_WEMPTY + ws), wp ^ 1);        // local: multicast commit of the MMAs (of every pair) that read it
                if (quad) {                                           // own quarter + the counterpart's quarter land here
                    mbar_expect_tx(bar(B_WFULL + ws), kWStage);
                    full_l = bar(B_WFULL + ws);
                } else {
                    if (hb == 0) mbar_expect_tx(bar(B_WFULL + ws), 2 * kWStage);
                    full_l = mapa_rank(bar(B_WFULL + ws), leader);
                }
                return base + offW + uint32_t(ws) * kWStage;
            };
            auto w_next = [&]() { if (++ws == NS) { ws = 0; wp ^= 1; } };
            auto load_w1 = [&](int c) {                               // rows c*128 + rank*64 .. +63 of W1, 4 k slabs of 8 KB
                uint32_t full_l;
                const uint32_t dst = w_slot(full_l);
                if (quad) {                                           // k slabs 2 pc, 2 pc + 1 of this half, to both pairs
                    for (int s = 2 * int(pc); s < 2 * int(pc) + 2; ++s)
                        tma_load_2d_mcast(dst + uint32_t(s) * (kSlab / 2), &tm_w1h, full_l, s * 64, c * kHC + int(hb) * 64, mc_mask);
                } else {
                    for (int s = 0; s < 4; ++s) tma_load_2d_pair(dst + uint32_t(s) * (kSlab / 2), &tm_w1h, full_l, s * 64, c * kHC + int(hb) * 64);
                }
                w_next();
            };
            auto load_w2 = [&](int c) {                               // rows rank*128 .. +127 of W2, k slabs c*128 + {0, 64}
                uint32_t full_l;
                const uint32_t dst = w_slot(full_l);
                if (quad) tma_load_2d_mcast(dst + pc * kSlab, &tm_w2h, full_l, c * kHC + int(pc) * 64, int(hb) * 128, mc_mask);
                else for (int j = 0; j < 2; ++j) tma_load_2d_pair(dst + uint32_t(j) * kSlab, &tm_w2h, full_l, c * kHC + j * 64, int(hb) * 128);
                w_next();
            };
            for (int j = 0; j < rounds; ++j) {
                load_w1(0);
                if (!TMH && NC > 1) load_w1(1);
                for (int c = 0; c < NC; ++c) {                     // the order the MMA warp consumes them in
                    if (c + (TMH ? 1 : 2) < NC) load_w1(c + (TMH ? 1 : 2));
                    load_w2(c);
                }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer: leader CTA only =====================
        if (hb == 0 && elect_one()) {
            const uint32_t idesc1 = umma_idesc_bf16(2 * kTM, kHC), idesc2 = umma_idesc_bf16(2 * kTM, kC);
            const uint32_t hi = uint32_t(1024 >> 4) | (1u << 14) | (2u << 29);
            auto lo = [](uint32_t addr) { return ((addr & 0x3FFFFu) >> 4) | (1u << 16); };
            const uint32_t a_lo = lo(base + kOffA), hs_lo = lo(base + kOffHs), w_lo = lo(base + offW);
            const uint32_t o_acc = tmem_base, h_acc = tmem_base + kC;
            int ws = 0; uint32_t wp = 0;
            uint32_t ph_hs = 0;
            auto w_wait = [&]() {                                     // (two pairs: both CTAs' relay warps have seen their halves land)
                mbar_wait_cluster(bar((quad ? B_PFULL : B_WFULL) + ws), wp);
                tc_fence_after();
                return w_lo + uint32_t(ws) * (kWStage >> 4);
            };
            auto w_release = [&]() { umma2_commit_mask(bar(B_WEMPTY + ws), all_mask); if (++ws == NS) { ws = 0; wp ^= 1; } };
            auto gemm1 = [&](int c) {
                const int b = c & 1;
                // Hacc[b] is released by GEMM2(c-2), in issue order (the tensor pipe executes in order)
                const uint32_t d = h_acc + uint32_t(b) * kHC;
                const uint32_t w = w_wait();
#pragma unroll
                for (int s = 0; s < 4; ++s)
#pragma unroll
                    for (int k = 0; k < 4; ++k)
                        umma2_bf16_lh(d, a_lo + uint32_t(s) * (kSlab >> 4) + 2 * k, hi, w + uint32_t(s) * (kSlab >> 5) + 2 * k, hi, idesc1,
                                      uint32_t(s | k));
                w_release();
                umma2_commit_mask(bar(B_HACC_FULL + b), pair_mask);
            };
            int it = 0;
            for (; it < rounds; ++it) {
                mbar_wait_cluster(bar(B_AFULL), it & 1);
                tc_fence_after();
                constexpr int LA = TMH ? 1 : 2;                           // GEMM1 lookahead (chunks)
                gemm1(0);
                if (LA == 2 && NC > 1) gemm1(1);
                if (NC <= LA) umma2_commit_mask(bar(B_AEMPTY), pair_mask);
                for (int c = 0; c < NC; ++c) {
                    if (c + LA < NC) {
                        gemm1(c + LA);
                        if (c + LA + 1 == NC) umma2_commit_mask(bar(B_AEMPTY), pair_mask);
                    }
                    const int b = c & 1;
                    const uint32_t hs_par = (ph_hs >> b) & 1;
                    ph_hs ^= 1u << b;
                    uint32_t w = 0;
                    // GEMM2(c) in four steps of K = 32: step q is issued as soon as the GELU warps have stored hidden columns
                    // [32 q, 32 q + 32) -- the first MMAs run while the rest of the chunk is still in the GELU
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        mbar_wait_cluster(bar(B_HS_FULL + 4 * b + q), hs_par);
                        if (q == 0) {
                            if (c == 0) mbar_wait_cluster(bar(B_OEMPTY), (it & 1) ^ 1);
                            w = w_wait();
                        }
                        tc_fence_after();
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            const int kk = 2 * q + e, j = kk >> 2, k = kk & 3;     // K slice kk = hidden columns [16 kk, +16)
                            // hidden 32 q + 16 e .. +15 = 8 packed columns at Hacc[b] + 32 q + 8 e: a GELU warp packs the 32 hidden
                            // columns of a sub-step into the first 16 of the fp32 columns it read
                            umma2_bf16_ts(o_acc, h_acc + uint32_t(b) * kHC + uint32_t(32 * q + 8 * e), w + uint32_t(j) * (kSlab >> 4) + 2 * k, hi,
                                          idesc2, uint32_t(c | kk));
                        }
                    }
                    w_release();
                }
                umma2_commit_mask(bar(B_OFULL), pair_mask);
            }
        }
    } else if (warp == 15) {
        // ===================== input-tile producer (both CTAs): own d tile.  A thread of its own: behind the weight loads in one
        // program order, a pair waiting for its A buffer would hold back the weight quarters the OTHER pair of the cluster needs.
        if (elect_one()) {
            const uint32_t afull_l = mapa_rank(bar(B_AFULL), leader);     // the leader's barrier, as a cluster address
            uint32_t ap = 0;
            for (int j = 0; j < rounds; ++j) {
                const int tile = 2 * (pair0 + j * n_pairs) + int(hb);  // past n_tiles: an all-padding tile (zero-filled by TMA)
                mbar_wait(bar(B_AEMPTY), ap ^ 1);
                if (hb == 0) mbar_expect_tx(bar(B_AFULL), 2 * 4 * kSlab);
                for (int s = 0; s < 4; ++s) tma_load_2d_pair(base + kOffA + s * kSlab, &tm_d, afull_l, s * 64, tile * kTM);
                ap ^= 1;
            }
        }
    } else if (warp == 14) {
        // ===================== relay (clusters of two pairs): this CTA's half of a weight stage has landed -> tell the pair's leader ====
        // A multicast TMA signals the barrier at the same offset in each destination CTA, so the leader cannot be told directly.
        if (quad && lane == 0) {
            const uint32_t pfull_l = mapa_rank(bar(B_PFULL), leader);
            int ws = 0; uint32_t wp = 0;
            const int uses = rounds * 2 * NC;
            for (int u = 0; u < uses; ++u) {
                mbar_wait_cluster(bar(B_WFULL + ws), wp);
                mbar_arrive_cluster(pfull_l + 8u * uint32_t(ws));          // (relaxed: the bytes are in shared memory before the barrier flips)
                if (++ws == NS) { ws = 0; wp ^= 1; }
            }
        }
    } else {
        // ===================== epilogue warps (both CTAs) =====================
        // Warps 2..5: GELU, one per TMEM lane quadrant = one per scheduler.  Warps 6..13: output drain, two per quadrant.
        // Why two kinds: clock64 around the phases showed the epilogue as ONE serial resource per scheduler -- the GELU of
        // the next tile's first chunks waited for the previous tile's drain, and GEMM2(c) for the slowest of 32 warps.
        // Now the GELU warp of a scheduler walks a chunk in four 32-column sub-steps and signals each (GEMM2's first MMAs are
        // issued a quarter of the way through), the MUFU pipe -- the floor of this phase: one MUFU.TANH per element at 4
        // lanes per clock = 1024 cycles per chunk -- is fed by one instruction stream, and the drain runs beside it.
        const int quad = warp & 3;
        const int r = quad * 32 + lane;
        const uint32_t t_lane = tmem_base + (uint32_t(quad * 32) << 16);
        if (warp < 6) {
            const uint32_t hs_full_l = mapa_rank(bar(B_HS_FULL), leader);
            uint32_t ph_use = 0;
            for (int j = 0; j < rounds; ++j) {
                for (int c = 0; c < NC; ++c) {
                    const int b = c & 1;
                    mbar_wait(bar(B_HACC_FULL + b), (ph_use >> b) & 1);
                    ph_use ^= 1u << b;
                    tc_fence_after();
                    const uint32_t hbase = t_lane + kC + uint32_t(b) * kHC;
                    uint32_t va[32], vb[32];
                    tmem_ld32_nowait(hbase, va);
                    auto sub = [&](const uint32_t (&v)[32], int q) {
                        uint32_t pk[16];
#pragma unroll
                        for (int j = 0; j < 32; j += 2) {                 // half biases from the constant bank: warp-uniform address
                            const float *hb = p.hb1v + c * kHC + q * 32 + j;
                            pk[j / 2] = gelu_bias2_pk(__uint_as_float(v[j]), __uint_as_float(v[j + 1]), hb[0], hb[1]);
                        }
                        // the 32 hidden columns of the sub-step go, packed, over the first 16 of the fp32 columns just read
                        tmem_st16(hbase + uint32_t(q * 32), pk);
                        tmem_st_wait();
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive_cluster(hs_full_l + 8u * uint32_t(4 * b + q));
                    };
                    // the load of sub-step q + 1 is in flight while sub-step q is computed
                    tmem_ld_wait(); tmem_ld32_nowait(hbase + 32, vb); sub(va, 0);
                    tmem_ld_wait(); tmem_ld32_nowait(hbase + 64, va); sub(vb, 1);
                    tmem_ld_wait(); tmem_ld32_nowait(hbase + 96, vb); sub(va, 2);
                    tmem_ld_wait(); sub(vb, 3);
                }
            }
        } else {
            const int half = (warp - 6) >> 2;                            // output columns [128 half, +128)
            const uint32_t oempty_l = mapa_rank(bar(B_OEMPTY), leader);
            for (int it = 0; it < rounds; ++it) {
                const int tile = 2 * (pair0 + it * n_pairs) + int(hb);
                const long long row = (long long)tile * kTM + r;
                const bool inb = row < p.n_px;
                // residual row segment (128 columns = 8 x 32 B), fetched BEFORE the wait for the last GEMM2s.  A thread is a
                // pixel row (TMEM lane), so every lane touches its own 32-byte sector: 256-bit accesses halve the L1 wavefronts.
                uint32_t res[8][8];
                {
                    const bf16 *rs = p.x + row * kC + half * 128;
#pragma unroll
                    for (int g = 0; g < 8; ++g) {
                        if (inb) ld_global_256(rs + 16 * g, res[g]);
                        else {
#pragma unroll
                            for (int e = 0; e < 8; ++e) res[g][e] = 0u;
                        }
                    }
                }
                mbar_wait(bar(B_OFULL), it & 1);
                tc_fence_after();
                // Oacc is single-buffered: the next tile's first GEMM2 waits until it is in registers.  Two loads in flight at
                // a time; the accumulator is RELEASED as soon as the last load has landed.
                uint32_t va[32], vb[32];
                auto emit = [&](const uint32_t (&vq)[32], int q) {
                    const int c0 = half * 128 + q * 32;
                    bf16 *dst = p.out + row * kC + c0;
#pragma unroll
                    for (int g = 0; g < 2; ++g) {                         // 16 columns = one 32-byte sector
                        uint32_t o8[8];
#pragma unroll
                        for (int e = 0; e < 8; ++e) {
                            const uint32_t xr = res[q * 2 + g][e];        // bf16 pair -> fp32: low half << 16, high half masked
                            const float *bc = p.b2v + c0 + g * 16 + 2 * e;      // (warp-uniform address, constant bank)
                            o8[e] = pack_bf16x2(__uint_as_float(vq[g * 16 + 2 * e]) + bc[0] + __uint_as_float(xr << 16),
                                                __uint_as_float(vq[g * 16 + 2 * e + 1]) + bc[1] + __uint_as_float(xr & 0xFFFF0000u));
                        }
                        if (inb) st_global_256(dst + 16 * g, o8);
                    }
                };
                tmem_ld32_nowait(t_lane + uint32_t(half * 128), va);
                tmem_ld32_nowait(t_lane + uint32_t(half * 128 + 32), vb);
                tmem_ld_wait();
                emit(va, 0);
                tmem_ld32_nowait(t_lane + uint32_t(half * 128 + 64), va);
                emit(vb, 1);
                tmem_ld32_nowait(t_lane + uint32_t(half * 128 + 96), vb);
                tmem_ld_wait();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(oempty_l);             // Oacc is in registers: the next tile may accumulate
                emit(va, 2);
                emit(vb, 3);
                __syncwarp();
                // tail filling: the depthwise kernel of the next trunk block polls these counters instead of waiting for the
                // whole grid (the __syncwarp above orders every lane's stores before lane 0's release)
                if (p.tile_done && lane == 0 && tile < p.n_tiles) asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(p.tile_done + tile) : "memory");
            }
        }
    }

    tc_fence_before();
    cluster_sync_all();                                              // both CTAs are done with TMEM and with each other's barriers
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512u) : "memory");
    }
}

}  // namespace

// ---------------------------------------------------------------- host side ----------------------------------
bool trunk_fusable(const ConvLayer &pw1, const ConvLayer &pw2)
{
    return pw1.c_in == kC && pw2.n == kC && pw2.n_pad == kC && pw1.n == pw2.c_in && pw1.n_pad == pw1.n && pw1.n % kHC == 0 && pw1.n <= kMaxHidden &&
           pw1.taps == 1 && pw2.taps == 1 && pw1.groups == 1 && pw2.groups == 1;
}

bool trunk_make_maps(TrunkMaps &m, const bf16 *d_base, long long n_px, const ConvLayer &pw1, const ConvLayer &pw2, std::string &err)
{
    m.ok = false;
    if (!trunk_fusable(pw1, pw2)) return true;
    // d: [n_px][256] bf16, box {64 ch, 128 px}; rows past n_px are zero-filled by TMA (ragged last tile)
    if (!tc_encode_2d(&m.tm_d, d_base, kC, (unsigned long long)n_px, 64, kTM, err)) return false;
    // W1: [hidden][256] (n rows, k contiguous), box {64, 128}; W2: [256][hidden], box {64, 256}
    if (!tc_encode_2d(&m.tm_w1, pw1.w, kC, (unsigned long long)pw1.n, 64, kHC, err)) return false;
    if (!tc_encode_2d(&m.tm_w2, pw2.w, (unsigned long long)pw2.c_in, kC, 64, kC, err)) return false;
    // CTA-pair kernel: each CTA loads half of every weight tile (64 of the 128 W1 rows, 128 of the 256 W2 rows)
    if (!tc_encode_2d(&m.tm_w1h, pw1.w, kC, (unsigned long long)pw1.n, 64, kHC / 2, err)) return false;
    if (!tc_encode_2d(&m.tm_w2h, pw2.w, (unsigned long long)pw2.c_in, kC, 64, kC / 2, err)) return false;
    m.ok = true;
    return true;
}

bool trunk_counts_tiles(long long n_px, bool pair) { return pair && (n_px + kTM - 1) / kTM >= 2; }

cudaError_t configure_trunk_kernels()
{
    cudaError_t e = cudaFuncSetAttribute(trunk_mlp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, int(kTrunkSmem));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(trunk_mlp_pair_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, int(kTrunkSmem));
    return e;
}

cudaError_t launch_trunk_mlp(const TrunkMaps &m, const ConvLayer &pw1, const ConvLayer &pw2, const bf16 *x, bf16 *out, long long n_px,
                             int num_sms, bool pair, LaunchStream st, uint32_t *tile_done, bool quad_clusters)
{
    TrunkParams p{};
    p.tile_done = tile_done;
    p.n_px = int(n_px);
    p.n_tiles = int((n_px + kTM - 1) / kTM);
    p.n_chunks = pw1.n / kHC;
    p.b1 = pw1.bias; p.b2 = pw2.bias;
    if (pw1.bias_host.size() >= size_t(pw1.n) && pw2.bias_host.size() >= size_t(kC) && pw1.n <= kMaxHidden) {
        for (int i = 0; i < pw1.n; ++i) p.hb1v[i] = 0.5f * pw1.bias_host[i];
        std::copy(pw2.bias_host.begin(), pw2.bias_host.begin() + kC, p.b2v);
    } else if (pair) {
        return cudaErrorInvalidValue;
    }
    p.x = x; p.out = out;
    if (pair && p.n_tiles >= 2) {
        const int n_ptiles = (p.n_tiles + 1) / 2;
        const int clusters = n_ptiles < num_sms / 2 ? n_ptiles : num_sms / 2;
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(unsigned(2 * clusters)); cfg.blockDim = dim3(kPairThreads); cfg.dynamicSmemBytes = kTrunkSmem; cfg.stream = st.s;
        cudaLaunchAttribute attr[3];
        unsigned na = 0;
        attr[na].id = cudaLaunchAttributeClusterDimension;
        attr[na].val.clusterDim.x = 2; attr[na].val.clusterDim.y = 1; attr[na].val.clusterDim.z = 1;
        ++na;
        if (quad_clusters && clusters % 2 == 0) {                   // two pairs per cluster where the GPC has room, one pair elsewhere
            attr[na].id = cudaLaunchAttributePreferredClusterDimension;
            attr[na].val.preferredClusterDim.x = 4; attr[na].val.preferredClusterDim.y = 1; attr[na].val.preferredClusterDim.z = 1;
            ++na;
        }
        if (st.pdl) {
            attr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
            attr[na].val.programmaticStreamSerializationAllowed = 1;
            ++na;
        }
        cfg.attrs = attr; cfg.numAttrs = na;
        return cudaLaunchKernelEx(&cfg, trunk_mlp_pair_kernel, m.tm_d, m.tm_w1h, m.tm_w2h, p);
    }
    const int grid = p.n_tiles < num_sms ? p.n_tiles : num_sms;
    return launch_pdl(trunk_mlp_kernel, grid, kTrunkThreads, kTrunkSmem, st, 1, m.tm_d, m.tm_w1, m.tm_w2, p);
}

}  // namespace ufnvc
