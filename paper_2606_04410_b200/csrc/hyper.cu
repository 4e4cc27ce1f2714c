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

__global__ void z_to_f64_kernel(const int16_t *__restrict__ z, double *__restrict__ out, int n_chunks, int c_z, int pz)
{
    asm volatile("griddepcontrol.wait;" ::: "memory");              // PDL: launched early, the predecessor's output is complete from here on
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    // z planar [n][c][pz] -> out NHWC [n][pz][c]
    const long long total = (long long)n_chunks * c_z * pz;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const int c = int(i % c_z);
        const long long r = i / c_z;
        const int p = int(r % pz);
        const int n = int(r / pz);
        out[i] = double(z[((long long)n * c_z + c) * pz + p]);
    }
}

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
// and k, 2 broadcast A vectors + 512 B of conflict-free B feed 512 DFMAs.  SPLIT = true: blockIdx.z = tap, raw partial
// sums go to part[tap][M][n_out] and hyper_reduce_kernel adds them in tap order (deterministic), for the two small
// layers that would otherwise occupy 16 CTAs.
constexpr int FM = 64, FN = 64, FK = 16, FPAD = 2;

template <bool SPLIT>
__global__ void __launch_bounds__(256) hyper_conv_fast_kernel(const double *__restrict__ in, const double *__restrict__ wt,
                                                              const double *__restrict__ bias, int n_img, int hz, int wz,
                                                              int c_in, int n_out, HyperEpi epi, double *__restrict__ part)
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

    const int tap_lo = SPLIT ? blockIdx.z : 0, tap_hi = SPLIT ? blockIdx.z + 1 : 9;
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
            if (SPLIT) {
                part[((long long)blockIdx.z * M + m) * n_out + o] = acc[i][j];
            } else {
                hyper_epilogue(epi, acc[i][j] + bias[o], m, o, pz, wz, n_out);
            }
        }
    }
}

__global__ void hyper_reduce_kernel(const double *__restrict__ part, const double *__restrict__ bias, double *__restrict__ out,
                                    long long MN, int n_out, const double *__restrict__ addend)
{
    asm volatile("griddepcontrol.wait;" ::: "memory");              // PDL: launched early, the predecessor's output is complete from here on
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < MN; i += (long long)gridDim.x * blockDim.x) {
        double v = part[i];
#pragma unroll
        for (int t = 1; t < 9; ++t) v += part[t * MN + i];                   // fixed tap order: run-to-run deterministic
        v += bias[i % n_out];
        v = v > 0.0 ? v : 0.0;
        if (addend) v += addend[i];                                          // s = x2 + q (R23)
        out[i] = v;
    }
}

cudaError_t launch_z_to_f64(const int16_t *z, double *out, int n_chunks, int c_z, int pz, LaunchStream st)
{
    const long long total = (long long)n_chunks * c_z * pz;
    const int blocks = int((total + 255) / 256 < 1184 ? (total + 255) / 256 : 1184);
    return launch_pdl(z_to_f64_kernel, unsigned(blocks), 256u, 0, st, 1, z, out, n_chunks, c_z, pz);
    return cudaGetLastError();
}

// same reduce, also emitting the 2-term bf16 split of the fp64 result: xs[m][o] = hi = bf16(v), xs[m][n_out + o] = bf16(v - hi),
// and xnorm2[m] = sum_o v^2 (fp32), the input of the head's a-priori error bound (decode.cu, R12).  One warp per
// z-pixel m, lanes stride the channels, fixed-order tree reduction: run-to-run deterministic.
__global__ void hyper_reduce_split_kernel(const double *__restrict__ part, const double *__restrict__ bias, double *__restrict__ out,
                                          bf16 *__restrict__ xs, float *__restrict__ xnorm2, long long M, int n_out,
                                          const double *__restrict__ addend)
{
    asm volatile("griddepcontrol.wait;" ::: "memory");              // PDL: launched early, the predecessor's output is complete from here on
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int lane = threadIdx.x & 31;
    const long long warps = ((long long)gridDim.x * blockDim.x) >> 5;
    const long long MN = M * n_out;
    for (long long m = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5; m < M; m += warps) {
        double ss = 0.0;
        for (int o = lane; o < n_out; o += 32) {
            const long long i = m * n_out + o;
            double v = part[i];
#pragma unroll
            for (int t = 1; t < 9; ++t) v += part[t * MN + i];               // fixed tap order
            v += bias[o];
            v = v > 0.0 ? v : 0.0;
            if (addend) v += addend[i];                                      // s = x2 + q (R23)
            out[i] = v;
            const bf16 hi = __double2bfloat16(v);
            const bf16 mid = __double2bfloat16(v - double(__bfloat162float(hi)));
            xs[m * 2 * n_out + o] = hi;
            xs[m * 2 * n_out + n_out + o] = mid;
            ss = fma(v, v, ss);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xFFFFFFFFu, ss, o);
        if (lane == 0) xnorm2[m] = float(ss);
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
        // lanes stride the channels; 4 independent accumulators (channel blocks) keep the fp64 pipe and the loads busy.
        // Fixed summation order per element -> run-to-run deterministic.
        double a4[4] = {0.0, 0.0, 0.0, 0.0};
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

cudaError_t launch_hyper_conv(const HyperLayer &L, const double *in, double *out, double *part, int n_img, int hz, int wz,
                              LaunchStream st, bf16 *xs, float *xnorm2, const double *addend)
{
    HyperEpi e{};
    e.mode = 0;
    e.out = out;
    const int M = n_img * hz * wz;
    if (fast_ok(L) && part) {                   // split over the 9 taps, then a deterministic reduce + bias + ReLU
        dim3 grid((M + FM - 1) / FM, (L.n + FN - 1) / FN, 9);
        if (cudaError_t le = launch_pdl_grid(hyper_conv_fast_kernel<true>, grid, 256u, st, in, L.w, L.bias, n_img, hz, wz, L.c_in, L.n, e, part)) return le;
        const long long MN = (long long)M * L.n;
        const int blocks = int((MN + 255) / 256 < 1184 ? (MN + 255) / 256 : 1184);
        if (xs) {
            const int wblocks = int(((long long)M * 32 + 255) / 256 < 1184 ? ((long long)M * 32 + 255) / 256 : 1184);
            if (cudaError_t le = launch_pdl(hyper_reduce_split_kernel, unsigned(wblocks), 256u, 0, st, 1, part, L.bias, out, xs, xnorm2, (long long)M, L.n, addend)) return le;
        }
        else if (cudaError_t le = launch_pdl(hyper_reduce_kernel, unsigned(blocks), 256u, 0, st, 1, part, L.bias, out, MN, L.n, addend)) return le;
        return cudaGetLastError();
    }
    if (addend || xs) return cudaErrorInvalidValue;       // the slow-shape kernel has no context branch (api.cu validates the shapes)
    dim3 grid((M + HM - 1) / HM, (L.n + HN - 1) / HN);
    hyper_conv_kernel<<<grid, 256, 0, st>>>(in, L.w, L.bias, n_img, hz, wz, L.c_in, L.n, e);
    return cudaGetLastError();
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
        if (cudaError_t le = launch_pdl_grid(hyper_conv_fast_kernel<false>, grid, 256u, st, in, L.w, L.bias, n_img, hz, wz, L.c_in, L.n, e, (double *)nullptr)) return le;
        return cudaGetLastError();
    }
    dim3 grid((M + HM - 1) / HM, (L.n + HN - 1) / HN);
    hyper_conv_kernel<<<grid, 256, 0, st>>>(in, L.w, L.bias, n_img, hz, wz, L.c_in, L.n, e);
    return cudaGetLastError();
}

}  // namespace ufnvc
