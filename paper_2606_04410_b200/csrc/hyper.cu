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
            const double v = acc[i][j] + bias[o];
            if (epi.mode == 0) {
                epi.out[(long long)m * n_out + o] = v > 0.0 ? v : 0.0;
            } else {
                // O2 / R14: pre-shuffle channel o = c2*16 + 4i + j at z-pixel (zy, zx) -> latent (4zy+i, 4zx+j), c2.
                const HeadParams &hp = epi.hp;
                const int img = m / pz, p = m % pz, zy = p / wz, zx = p % wz;
                const int c2 = o >> 4, ly = 4 * zy + ((o >> 2) & 3), lx = 4 * zx + (o & 3);
                if (ly >= hp.h || lx >= hp.w) continue;                        // crop [R2]
                if (c2 < hp.c_y) {
                    hp.mu[(((long long)img * hp.h + ly) * hp.w + lx) * hp.c_y + c2] = float(v);
                } else {
                    const long long e = (((long long)img * hp.h + ly) * hp.w + lx) * hp.c_y + (c2 - hp.c_y);
                    double u = v < hp.ln_lo ? hp.ln_lo : (v > hp.ln_hi ? hp.ln_hi : v);
                    // same operation order as the definition: floor((nb-1)*(u-lo)/(hi-lo) + 0.5), in double
                    const double t = floor(double(hp.n_buckets - 1) * (u - hp.ln_lo) / (hp.ln_hi - hp.ln_lo) + 0.5);
                    int k = int(t);
                    k = k < 0 ? 0 : (k > hp.n_buckets - 1 ? hp.n_buckets - 1 : k);
                    hp.idx[e] = uint8_t(k);
                    if (hp.lnscale) hp.lnscale[e] = float(u);
                }
            }
        }
    }
}

cudaError_t launch_z_to_f64(const int16_t *z, double *out, int n_chunks, int c_z, int pz, cudaStream_t st)
{
    const long long total = (long long)n_chunks * c_z * pz;
    const int blocks = int((total + 255) / 256 < 1184 ? (total + 255) / 256 : 1184);
    z_to_f64_kernel<<<blocks, 256, 0, st>>>(z, out, n_chunks, c_z, pz);
    return cudaGetLastError();
}

cudaError_t launch_hyper_conv(const HyperLayer &L, const double *in, double *out, int n_img, int hz, int wz,
                              cudaStream_t st)
{
    HyperEpi e{};
    e.mode = 0;
    e.out = out;
    dim3 grid((n_img * hz * wz + HM - 1) / HM, (L.n + HN - 1) / HN);
    hyper_conv_kernel<<<grid, 256, 0, st>>>(in, L.w, L.bias, n_img, hz, wz, L.c_in, L.n, e);
    return cudaGetLastError();
}

cudaError_t launch_hyper_head(const HyperLayer &L, const double *in, int n_img, int hz, int wz, const HeadParams &hp,
                              cudaStream_t st)
{
    HyperEpi e{};
    e.mode = 1;
    e.out = nullptr;
    e.hp = hp;
    dim3 grid((n_img * hz * wz + HM - 1) / HM, (L.n + HN - 1) / HN);
    hyper_conv_kernel<<<grid, 256, 0, st>>>(in, L.w, L.bias, n_img, hz, wz, L.c_in, L.n, e);
    return cudaGetLastError();
}

}  // namespace ufnvc
