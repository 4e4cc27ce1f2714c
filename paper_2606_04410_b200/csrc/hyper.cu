// A1 + A2: hyper-decoder -> per-element mean and scale-bucket index, in fp64.
// "our parameter estimation network ... simultaneously predicts the mean and the scales ... in a
// single forward pass".  Why fp64 (R12): the bucket index is an integer decided by a floating-point
// value; one flipped index desynchronises a whole rANS warp-stream, so the decision must be reproducible across
// implementations.  2.5 GMAC per 1080p chunk -- 0.3 % of the chunk's work -- so it runs on the FP64 pipe.
//
// Implicit GEMM on CUDA cores: M = z-pixels (all chunks), N = output channels, K = 9 taps x C_in.
// Block 256 threads = 16 x 16, tile 32 pixels x 64 channels, 2 x 4 outputs per thread, K step 16.
#include "ufnvc_internal.h"

namespace ufnvc {

constexpr int HM = 32, HN = 64, HK = 16;

struct HyperEpi {
    int mode;            // 0: ReLU -> NHWC double; 1: head
    double *out;
    HeadParams hp;
};

// ReLU -> NHWC double (mode 0), or the head (mode 1): O2 / R14 pixel-shuffle x4 + crop + split + clamp + bucket.
__device__ __forceinline__ void hyper_epilogue(const HyperEpi &epi, double v, int m, int o, int pz, int wz, int n_out)
{
    if (epi.mode == 0) {
        epi.out[(long long)m * n_out + o] = v > 0.0 ? v : 0.0;
        return;
    }
    // pre-shuffle channel o = c2*16 + 4i + j at z-pixel (zy, zx) -> latent (4zy+i, 4zx+j), channel c2.
    const HeadParams &hp = epi.hp;
    const int img = m / pz, p = m % pz, zy = p / wz, zx = p % wz;
    const int c2 = o >> 4, ly = 4 * zy + ((o >> 2) & 3), lx = 4 * zx + (o & 3);
    if (ly >= hp.h || lx >= hp.w) return;                                   // crop [R2]
    if (c2 < hp.c_y) {
        hp.mu[(((long long)img * hp.h + ly) * hp.w + lx) * hp.c_y + c2] = float(v);
    } else {
        const long long e = (((long long)img * hp.h + ly) * hp.w + lx) * hp.c_y + (c2 - hp.c_y);
        const double u = v < hp.ln_lo ? hp.ln_lo : (v > hp.ln_hi ? hp.ln_hi : v);
        // same operation order as the definition: floor((nb-1)*(u-lo)/(hi-lo) + 0.5), in double
        const double t = floor(double(hp.n_buckets - 1) * (u - hp.ln_lo) / (hp.ln_hi - hp.ln_lo) + 0.5);
        int k = int(t);
        k = k < 0 ? 0 : (k > hp.n_buckets - 1 ? hp.n_buckets - 1 : k);
        hp.idx[e] = uint8_t(k);
        if (hp.lnscale) hp.lnscale[e] = float(u);
    }
}

__global__ void __launch_bounds__(256) hyper_conv_kernel(const double *__restrict__ in, const double *__restrict__ wt,
                                                         const double *__restrict__ bias, int n_img, int hz, int wz,
                                                         int c_in, int n_out, HyperEpi epi)
{
    __shared__ double As[HK][HM + 1];
    __shared__ double Bs[HK][HN];
    const int pz = hz * wz;
    const int M = n_img * pz;
    const int m0 = blockIdx.x * HM, n0 = blockIdx.y * HN;
    const int tid = threadIdx.x, ty = tid / 16, tx = tid % 16;

    double acc[2][4] = {};
    // A loader: 32 pixels x 16 k -> 512 elements, 2 per thread; B loader: 16 k x 64 n -> 1024, 4 per thread.
    const int a_pix = tid / 8, a_k = (tid % 8) * 2;
    const int gm = m0 + a_pix;
    const int a_img = gm < M ? gm / pz : 0, a_p = gm < M ? gm % pz : 0;
    const int a_y = a_p / wz, a_x = a_p % wz;
    const int b_k = tid / 16, b_n = (tid % 16) * 4;

    for (int tap = 0; tap < 9; ++tap) {
        const int yy = a_y + tap / 3 - 1, xx = a_x + tap % 3 - 1;
        const bool a_ok = gm < M && yy >= 0 && yy < hz && xx >= 0 && xx < wz;
        const double *a_src = in + ((long long)a_img * pz + (long long)yy * wz + xx) * c_in;
        for (int k0 = 0; k0 < c_in; k0 += HK) {
            double a0 = 0.0, a1 = 0.0;
            if (a_ok) {
                if (k0 + a_k < c_in) a0 = a_src[k0 + a_k];
                if (k0 + a_k + 1 < c_in) a1 = a_src[k0 + a_k + 1];
            }
            As[a_k][a_pix] = a0;
            As[a_k + 1][a_pix] = a1;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                double b = 0.0;
                if (k0 + b_k < c_in && n0 + b_n + j < n_out)
                    b = wt[((long long)tap * c_in + k0 + b_k) * n_out + n0 + b_n + j];
                Bs[b_k][b_n + j] = b;
            }
            __syncthreads();
#pragma unroll
            for (int k = 0; k < HK; ++k) {
                const double av0 = As[k][ty * 2], av1 = As[k][ty * 2 + 1];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const double bv = Bs[k][tx * 4 + j];
                    acc[0][j] = fma(av0, bv, acc[0][j]);
                    acc[1][j] = fma(av1, bv, acc[1][j]);
                }
            }
            __syncthreads();
        }
    }

#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const int m = m0 + ty * 2 + i;
        if (m >= M) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int o = n0 + tx * 4 + j;
            if (o >= n_out) continue;
            hyper_epilogue(epi, acc[i][j] + bias[o], m, o, pz, wz, n_out);
        }
    }
}


// ---- fast path: 64 x 64 tile, 256 threads, 4 x 4 doubles per thread, K step 16, register-prefetch double buffering.
// Requires c_in % 16 == 0 (a K step never straddles a tap) and n_out % 4 == 0.  DFMA-pipe bound by design: per warp
// and k, 2 broadcast A vectors + 512 B of conflict-free B feed 512 DFMAs.  Used by the all-fp64 head (N = 4096 gives it
// enough blocks); layers 0 and 1 run on hyper_conv_direct_kernel below.
constexpr int FM = 64, FN = 64, FK = 16, FPAD = 2;

__global__ void __launch_bounds__(256) hyper_conv_fast_kernel(const double *__restrict__ in, const double *__restrict__ wt,
                                                              const double *__restrict__ bias, int n_img, int hz, int wz,
                                                              int c_in, int n_out, HyperEpi epi)
{
    __shared__ __align__(16) double As[2][FK][FM + FPAD];
    __shared__ __align__(16) double Bs[2][FK][FN];
    asm volatile("griddepcontrol.wait;" ::: "memory");              // PDL: launched early, the predecessor's output is complete from here on
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int pz = hz * wz;
    const int M = n_img * pz;
    const int m0 = blockIdx.x * FM, n0 = blockIdx.y * FN;
    const int tid = threadIdx.x, ty = tid >> 4, tx = tid & 15;

    // loaders: A 64 px x 16 k (4 consecutive k per thread), B 16 k x 64 n (4 consecutive n per thread)
    const int a_pix = tid >> 2, a_k = (tid & 3) * 4;
    const int gm = m0 + a_pix;
    const int a_img = gm < M ? gm / pz : 0, a_p = gm < M ? gm % pz : 0;
    const int a_y = a_p / wz, a_x = a_p % wz;
    const int b_k = tid >> 4, b_n = (tid & 15) * 4;
    const bool b_ok = n0 + b_n < n_out;

    const int tap_lo = 0, tap_hi = 9;
    const int ksteps_per_tap = c_in / FK;
    const int total_steps = (tap_hi - tap_lo) * ksteps_per_tap;

    double2 ra[2], rb[2];
    auto gload = [&](int step) {
        const int tap = tap_lo + step / ksteps_per_tap, k0 = (step % ksteps_per_tap) * FK;
        const int yy = a_y + tap / 3 - 1, xx = a_x + tap % 3 - 1;
        const bool a_ok = gm < M && yy >= 0 && yy < hz && xx >= 0 && xx < wz;
        ra[0] = ra[1] = make_double2(0.0, 0.0);
        if (a_ok) {
            const double2 *src = reinterpret_cast<const double2 *>(in + ((long long)a_img * pz + (long long)yy * wz + xx) * c_in + k0 + a_k);
            ra[0] = src[0]; ra[1] = src[1];
        }
        rb[0] = rb[1] = make_double2(0.0, 0.0);
        if (b_ok) {
            const double2 *src = reinterpret_cast<const double2 *>(wt + ((long long)tap * c_in + k0 + b_k) * n_out + n0 + b_n);
            rb[0] = src[0]; rb[1] = src[1];
        }
    };
    auto sstore = [&](int buf) {
        As[buf][a_k + 0][a_pix] = ra[0].x; As[buf][a_k + 1][a_pix] = ra[0].y;
        As[buf][a_k + 2][a_pix] = ra[1].x; As[buf][a_k + 3][a_pix] = ra[1].y;
        *reinterpret_cast<double2 *>(&Bs[buf][b_k][b_n]) = rb[0];
        *reinterpret_cast<double2 *>(&Bs[buf][b_k][b_n + 2]) = rb[1];
    };

    double acc[4][4] = {};
    gload(0);
    sstore(0);
    __syncthreads();
    for (int step = 0; step < total_steps; ++step) {
        const int buf = step & 1;
        if (step + 1 < total_steps) gload(step + 1);
#pragma unroll
        for (int k = 0; k < FK; ++k) {
            const double2 a01 = *reinterpret_cast<const double2 *>(&As[buf][k][ty * 4]);
            const double2 a23 = *reinterpret_cast<const double2 *>(&As[buf][k][ty * 4 + 2]);
            const double2 b01 = *reinterpret_cast<const double2 *>(&Bs[buf][k][tx * 2]);          // columns 2tx, 2tx+1
            const double2 b23 = *reinterpret_cast<const double2 *>(&Bs[buf][k][32 + tx * 2]);     // columns 32+2tx, 33+2tx
            const double a[4] = {a01.x, a01.y, a23.x, a23.y}, b[4] = {b01.x, b01.y, b23.x, b23.y};
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] = fma(a[i], b[j], acc[i][j]);
        }
        if (step + 1 < total_steps) sstore(buf ^ 1);
        __syncthreads();
    }

#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int m = m0 + ty * 4 + i;
        if (m >= M) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int o = n0 + (j < 2 ? tx * 2 + j : 32 + tx * 2 + (j - 2));
            if (o >= n_out) continue;
            hyper_epilogue(epi, acc[i][j] + bias[o], m, o, pz, wz, n_out);
        }
    }
}

// ---- layers 0 and 1 (O1): direct implicit GEMM in fp64 on the FP64 TENSOR cores (mma.sync m8n8k4), ONE launch per layer.
// The CUDA-core version of this kernel (2 x 2 outputs per thread, operands by LDS.128) took 27 + 16 us for 7 us of FP64 work
// (61 DFMA per clock and SM measured, the same rate as DMMA), and clock64 stamps around its K steps did not move with a warm L2:
// every LDS.128 delivers 512 bytes to a warp whatever the broadcast, 2 of them per 4 DFMA, and 16 warps saturate the 128 B/clk
// shared-memory port (2.6 k cycles per 16-k step).  The m8n8k4 fragments need ONE 8-byte load per thread and operand for 256
// FMAs of the warp: a fifth of the bytes (22 + 14 us).  What bounds it now is the operand traffic of so small a tile: 56 MB from
// L2 per layer-1 launch, fetched in bursts by 2048 warps at once (a step's loads take 6-7 k cycles to come back); an L2
// prefetch of the weights ahead of the predecessor wait changed nothing.
// The z map is tiny (510 pixels at 1080p), so the output tile is small -- 16 pixels x 32 channels, 32 x 4 blocks for 510 x 128 --
// and K (9 taps x C_in) is split over the block's 16 warps: each warp runs its share of the 16-k steps on its own shared-memory
// stage (global -> registers one step ahead -> shared, __syncwarp only) and holds the whole tile's partial sums (2 x 4 fragments);
// the partials are added in warp order at the end (deterministic).
// ZIN: the input is the int16 hyper-latent itself, planar [n][c_z][pz] (layer 0), converted on load.
// Epilogue: + bias, ReLU; layer 1 also adds the context branch q (R23), writes the 2-term bf16 split hi | mid the tensor-core
// head reads, and this block's share of sum_c v^2 per pixel (xnorm2[m][n-tile]; the head adds the shares in order).
constexpr int DM = 16, DN = 32, DK = 16, DW = 16;
constexpr int kAS = 20, kBS = 36;           // row strides (doubles) of the A [k][pixel] and B [k][n] stages: = 4 (mod 16), so the 16 8-byte
                                            // fragment loads of a half-warp (4 k rows x 4 columns) fall into 16 different bank pairs
constexpr int kStageD = DK * kAS + DK * kBS;                                  // 896 doubles per warp
constexpr size_t kDirectSmem = size_t(DW) * kStageD * sizeof(double);         // 112 KB: dynamic
static_assert(DM * DN <= kStageD, "a warp's partial tile fits its own stage");

__device__ __forceinline__ void dmma884(double (&d)[2], double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};" : "+d"(d[0]), "+d"(d[1]) : "d"(a), "d"(b));
}

template <bool ZIN>
__global__ void __launch_bounds__(32 * DW) hyper_conv_direct_kernel(const void *__restrict__ in_raw, const double *__restrict__ wt,
                                                                    const double *__restrict__ bias, int n_img, int hz, int wz, int c_in,
                                                                    int n_out, double *__restrict__ out, const double *__restrict__ addend,
                                                                    bf16 *__restrict__ xs, float *__restrict__ xnorm2)
{
    extern __shared__ __align__(16) double direct_smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // (the bias does not depend on the predecessor grid: requested before the wait for it)
    const double bias_o = blockIdx.y * DN + lane < n_out ? bias[blockIdx.y * DN + lane] : 0.0;
    asm volatile("griddepcontrol.wait;" ::: "memory");              // PDL: launched early, the predecessor's output is complete from here on
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    double *As = direct_smem + size_t(warp) * kStageD, *Bs = As + DK * kAS;
    const int pz = hz * wz;
    const int M = n_img * pz;
    const int m0 = blockIdx.x * DM, n0 = blockIdx.y * DN;
    // loaders (per warp): A 16 px x 16 k (8 consecutive k per lane), B 16 k x 32 n (16 consecutive n per lane)
    const int a_pix = lane >> 1, a_k = (lane & 1) * 8;
    const int gm = m0 + a_pix;
    const int a_img = gm < M ? gm / pz : 0, a_p = gm < M ? gm % pz : 0;
    const int a_y = a_p / wz, a_x = a_p % wz;
    const int b_k = lane >> 1, b_n = (lane & 1) * 16;
    const bool b_ok = n0 + b_n < n_out;                             // n_out % 16 == 0
    const int ksteps_per_tap = c_in / DK;
    const int total_steps = 9 * ksteps_per_tap;
    const int s_lo = total_steps * warp / DW, s_hi = total_steps * (warp + 1) / DW;   // this warp's K steps
    const double *in = static_cast<const double *>(in_raw);
    const int16_t *zin = static_cast<const int16_t *>(in_raw);

    double ra[8];
    double2 rb[8];
    auto gload = [&](int step) {
        const int tap = step / ksteps_per_tap, k0 = (step % ksteps_per_tap) * DK;
        const int yy = a_y + tap / 3 - 1, xx = a_x + tap % 3 - 1;
#pragma unroll
        for (int j = 0; j < 8; ++j) ra[j] = 0.0;
        if (gm < M && yy >= 0 && yy < hz && xx >= 0 && xx < wz) {
            if (ZIN) {
                const int16_t *src = zin + ((long long)a_img * c_in + k0 + a_k) * pz + (long long)yy * wz + xx;
#pragma unroll
                for (int j = 0; j < 8; ++j) ra[j] = double(src[(long long)j * pz]);
            } else {
                const double2 *src = reinterpret_cast<const double2 *>(in + ((long long)a_img * pz + (long long)yy * wz + xx) * c_in + k0 + a_k);
#pragma unroll
                for (int j = 0; j < 4; ++j) { const double2 v = src[j]; ra[2 * j] = v.x; ra[2 * j + 1] = v.y; }
            }
        }
#pragma unroll
        for (int j = 0; j < 8; ++j) rb[j] = make_double2(0.0, 0.0);
        if (b_ok) {
            const double2 *src = reinterpret_cast<const double2 *>(wt + ((long long)tap * c_in + k0 + b_k) * n_out + n0 + b_n);
#pragma unroll
            for (int j = 0; j < 8; ++j) rb[j] = src[j];
        }
    };
    auto sstore = [&]() {
#pragma unroll
        for (int j = 0; j < 8; ++j) As[(a_k + j) * kAS + a_pix] = ra[j];
#pragma unroll
        for (int j = 0; j < 8; ++j) *reinterpret_cast<double2 *>(&Bs[b_k * kBS + b_n + 2 * j]) = rb[j];
    };

    double acc[2][4][2] = {};                                       // fragment (mt, nt): rows 8 mt + lane / 4, columns 8 nt + 2 (lane % 4) + {0, 1}
    const int fk = lane & 3, fr = lane >> 2;
    if (s_lo < s_hi) gload(s_lo);
    for (int step = s_lo; step < s_hi; ++step) {
        __syncwarp();                                               // the previous step's fragment loads are done
        sstore();
        __syncwarp();
        if (step + 1 < s_hi) gload(step + 1);
#pragma unroll
        for (int k4 = 0; k4 < DK / 4; ++k4) {
            double a[2], b[4];
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) a[mt] = As[(4 * k4 + fk) * kAS + 8 * mt + fr];
#pragma unroll
            for (int nt = 0; nt < 4; ++nt) b[nt] = Bs[(4 * k4 + fk) * kBS + 8 * nt + fr];
#pragma unroll
            for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                for (int nt = 0; nt < 4; ++nt) dmma884(acc[mt][nt], a[mt], b[nt]);
        }
    }
    // fixed-order reduction over the warps: every warp parks its partial tile [pixel][channel] in its own (now idle) stage
    __syncwarp();
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
        for (int nt = 0; nt < 4; ++nt)
            *reinterpret_cast<double2 *>(&As[(8 * mt + fr) * DN + 8 * nt + 2 * fk]) = make_double2(acc[mt][nt][0], acc[mt][nt][1]);
    __syncthreads();
    // one output per thread: warp = pixel of the tile, lane = channel
    const int m = m0 + warp, o = n0 + lane;
    double v = 0.0;
#pragma unroll
    for (int w2 = 0; w2 < DW; ++w2) v += direct_smem[size_t(w2) * kStageD + warp * DN + lane];
    double ss = 0.0;
    if (m < M && o < n_out) {
        v += bias_o;
        v = v > 0.0 ? v : 0.0;
        const long long e = (long long)m * n_out + o;
        if (addend) v += addend[e];                                 // s = x2 + q (R23)
        out[e] = v;
        if (xs) {
            const bf16 hi = __double2bfloat16(v);
            xs[(long long)m * 2 * n_out + o] = hi;
            xs[(long long)m * 2 * n_out + n_out + o] = __double2bfloat16(v - double(__bfloat162float(hi)));
        }
        ss = v * v;
    }
    if (xnorm2) {                                                   // the warp holds pixel m's 32 channels of this n tile
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) ss += __shfl_xor_sync(0xFFFFFFFFu, ss, d);
        if (lane == 0 && m < M) xnorm2[(long long)m * gridDim.y + blockIdx.y] = float(ss);
    }
}

// Exact fp64 re-evaluation of ln sigma for the flagged elements: one warp per element, lanes stride the channels,
// fixed-order tree reduction (deterministic).  list[i] = element index in [n][h][w][c_y].
__global__ void __launch_bounds__(256) hyper_fix_kernel(const uint32_t *__restrict__ list, const uint32_t *__restrict__ count,
                                                        const double *__restrict__ x2, const double *__restrict__ fix_w,
                                                        const double *__restrict__ fix_b, int c_h, int hz, int wz, HeadParams hp)
{
    const int lane = threadIdx.x & 31;
    asm volatile("griddepcontrol.wait;" ::: "memory");              // PDL: the head conv has written the list and its count
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); // the rANS blocks may start loading their tables
    const unsigned n = *count;
    const unsigned warps = (gridDim.x * blockDim.x) >> 5;
    for (unsigned i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; i < n; i += warps) {
        const unsigned e = list[i];
        const int c2 = int(e % unsigned(hp.c_y));
        unsigned r = e / unsigned(hp.c_y);
        const int lx = int(r % unsigned(hp.w)); r /= unsigned(hp.w);
        const int ly = int(r % unsigned(hp.h));
        const int img = int(r / unsigned(hp.h));
        const int zy = ly >> 2, zx = lx >> 2, ij = ((ly & 3) << 2) | (lx & 3);
        const double *wrow = fix_w + (size_t(c2) * 16 + ij) * 9 * c_h;
        // lanes stride the channels.  The kernel is bound by the latency of its loads (x patch and weight row come from L2),
        // not by the 1152 DFMAs of an element: all loads of THREE taps are issued before their FMAs (24 in flight per lane
        // for c_h = 128; one tap at a time measured 1.4x slower).  Four accumulators, fixed summation order per element ->
        // run-to-run deterministic.
        double a4[4] = {0.0, 0.0, 0.0, 0.0};
        if (c_h == 128) {
#pragma unroll
            for (int t3 = 0; t3 < 9; t3 += 3) {
                double xv[3][4], wv[3][4];
#pragma unroll
                for (int t = 0; t < 3; ++t) {
                    const int tap = t3 + t;
                    const int yy = zy + tap / 3 - 1, xx = zx + tap % 3 - 1;
                    const bool ok = yy >= 0 && yy < hz && xx >= 0 && xx < wz;
                    const double *xr = x2 + ((size_t(img) * hz + (ok ? yy : zy)) * wz + (ok ? xx : zx)) * c_h;
                    const double *wr = wrow + tap * c_h;
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        xv[t][u] = ok ? xr[lane + 32 * u] : 0.0;
                        wv[t][u] = wr[lane + 32 * u];
                    }
                }
#pragma unroll
                for (int t = 0; t < 3; ++t)
#pragma unroll
                    for (int u = 0; u < 4; ++u) a4[u] = fma(xv[t][u], wv[t][u], a4[u]);
            }
        } else {
#pragma unroll
            for (int tap = 0; tap < 9; ++tap) {
                const int yy = zy + tap / 3 - 1, xx = zx + tap % 3 - 1;
                if (yy < 0 || yy >= hz || xx < 0 || xx >= wz) continue;
                const double *xr = x2 + ((size_t(img) * hz + yy) * wz + xx) * c_h;
                const double *wr = wrow + tap * c_h;
                int c = lane;
                for (; c + 96 < c_h; c += 128) {
#pragma unroll
                    for (int u = 0; u < 4; ++u) a4[u] = fma(xr[c + 32 * u], wr[c + 32 * u], a4[u]);
                }
                for (; c < c_h; c += 32) a4[0] = fma(xr[c], wr[c], a4[0]);
            }
        }
        double acc = (a4[0] + a4[1]) + (a4[2] + a4[3]);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xFFFFFFFFu, acc, o);
        if (lane == 0) {
            const double v = acc + fix_b[size_t(c2) * 16 + ij];
            const double u = v < hp.ln_lo ? hp.ln_lo : (v > hp.ln_hi ? hp.ln_hi : v);
            const double t = floor(double(hp.n_buckets - 1) * (u - hp.ln_lo) / (hp.ln_hi - hp.ln_lo) + 0.5);
            int k = int(t);
            k = k < 0 ? 0 : (k > hp.n_buckets - 1 ? hp.n_buckets - 1 : k);
            hp.idx[e] = uint8_t(k);
            if (hp.lnscale) hp.lnscale[e] = float(u);
        }
    }
}

static bool fast_ok(const HyperLayer &L) { return L.c_in % FK == 0 && L.n % 4 == 0; }

cudaError_t configure_hyper_kernels()
{
    cudaError_t e = cudaFuncSetAttribute(hyper_conv_direct_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(kDirectSmem));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(hyper_conv_direct_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(kDirectSmem));
    return e;
}

template <typename... KArgs, typename... Args>
static cudaError_t launch_direct(void (*kern)(KArgs...), dim3 grid, LaunchStream st, Args &&...args)      // 2-D grid + dynamic smem + PDL
{
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid; cfg.blockDim = dim3(32 * DW); cfg.dynamicSmemBytes = kDirectSmem; cfg.stream = st.s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = st.pdl ? 1u : 0u;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

int hyper_xnorm_parts(const HyperLayer &L) { return (L.n + DN - 1) / DN; }

cudaError_t launch_hyper_conv(const HyperLayer &L, const void *in, bool in_is_z, double *out, int n_img, int hz, int wz, LaunchStream st,
                              bf16 *xs, float *xnorm2, const double *addend)
{
    const int M = n_img * hz * wz;
    if (L.c_in % DK == 0 && L.n % 16 == 0) {
        dim3 grid((M + DM - 1) / DM, (L.n + DN - 1) / DN);
        if (in_is_z)
            return launch_direct(hyper_conv_direct_kernel<true>, grid, st, in, L.w, L.bias, n_img, hz, wz, L.c_in, L.n, out, addend, xs, xnorm2);
        return launch_direct(hyper_conv_direct_kernel<false>, grid, st, in, L.w, L.bias, n_img, hz, wz, L.c_in, L.n, out, addend, xs, xnorm2);
    }
    return cudaErrorInvalidValue;         // api.cu validates c_z % 16 == 0, c_hyper % 16 == 0
}

// ---- R23: q = ReLU(W_p pool4(C) + b_p), the context branch of the prior input, in fp64.  The context is a bf16 tensor (its
// values are exact in fp64 and so are the 16-term sums), so both sides of the parity test evaluate the same real numbers up
// to the order of a 256-term fp64 sum.  One block per z-pixel: pool into shared memory, then thread o = output channel.
__global__ void __launch_bounds__(128) ctx_prior_kernel(const bf16 *__restrict__ ctx, int stride, int c_ctx, const double *__restrict__ w_p,
                                                        const double *__restrict__ b_p, double *__restrict__ q, int h, int w, int hz, int wz,
                                                        int c_h)
{
    extern __shared__ double pool[];                                 // [c_ctx]
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int m = blockIdx.x, pz = hz * wz;
    const int img = m / pz, r = m % pz, zy = r / wz, zx = r % wz;
    for (int k = threadIdx.x; k < c_ctx; k += blockDim.x) {
        double s = 0.0;
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int y = 4 * zy + i, x = 4 * zx + j;
                if (y < h && x < w) s += double(__bfloat162float(ctx[(((long long)img * h + y) * w + x) * stride + k]));
            }
        pool[k] = s / 16.0;
    }
    __syncthreads();
    for (int o = threadIdx.x; o < c_h; o += blockDim.x) {
        double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;               // fixed summation order: deterministic
        int k = 0;
        for (; k + 3 < c_ctx; k += 4) {
            a0 = fma(w_p[(long long)k * c_h + o], pool[k], a0);
            a1 = fma(w_p[(long long)(k + 1) * c_h + o], pool[k + 1], a1);
            a2 = fma(w_p[(long long)(k + 2) * c_h + o], pool[k + 2], a2);
            a3 = fma(w_p[(long long)(k + 3) * c_h + o], pool[k + 3], a3);
        }
        for (; k < c_ctx; ++k) a0 = fma(w_p[(long long)k * c_h + o], pool[k], a0);
        const double v = (a0 + a1) + (a2 + a3) + b_p[o];
        q[(long long)m * c_h + o] = v > 0.0 ? v : 0.0;
    }
}

cudaError_t launch_ctx_prior(const bf16 *ctx, int stride, int c_ctx, const double *w_p, const double *b_p, double *q, int n_img, int h, int w,
                             int hz, int wz, int c_h, LaunchStream st)
{
    return launch_pdl(ctx_prior_kernel, unsigned(n_img * hz * wz), 128u, size_t(c_ctx) * 8, st, 1, ctx, stride, c_ctx, w_p, b_p, q, h, w, hz, wz, c_h);
}

cudaError_t launch_hyper_fix(const uint32_t *list, const uint32_t *count, const double *x2, const double *fix_w, const double *fix_b,
                             int c_h, int hz, int wz, const HeadParams &hp, int num_sms, LaunchStream st)
{
    return launch_pdl(hyper_fix_kernel, unsigned(num_sms * 4), 256u, 0, st, 1, list, count, x2, fix_w, fix_b, c_h, hz, wz, hp);
}

cudaError_t launch_hyper_head(const HyperLayer &L, const double *in, int n_img, int hz, int wz, const HeadParams &hp,
                              LaunchStream st)
{
    HyperEpi e{};
    e.mode = 1;
    e.out = nullptr;
    e.hp = hp;
    const int M = n_img * hz * wz;
    if (fast_ok(L)) {
        dim3 grid((M + FM - 1) / FM, (L.n + FN - 1) / FN);
        if (cudaError_t le = launch_pdl_grid(hyper_conv_fast_kernel, grid, 256u, st, in, L.w, L.bias, n_img, hz, wz, L.c_in, L.n, e)) return le;
        return cudaGetLastError();
    }
    dim3 grid((M + HM - 1) / HM, (L.n + HN - 1) / HN);
    hyper_conv_kernel<<<grid, 256, 0, st>>>(in, L.w, L.bias, n_img, hz, wz, L.c_in, L.n, e);
    return cudaGetLastError();
}

}  // namespace ufnvc
