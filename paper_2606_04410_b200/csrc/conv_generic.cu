// CUDA-core implicit-GEMM convolution (any channel count that is a multiple of 8) and the depthwise 3x3.
// The generic conv serves the shapes the tcgen05 kernel does not take (config 1's 48/32/16-channel layers) and is
// the on-device cross-check of the tensor-core path.  Activations NHWC bf16, fp32 accumulate.
//   out[pix][n] = bias[n] + sum_{tap, c} in[pix + tap][c] * w[group][tap][n][c]
#include "epilogue.cuh"
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

cudaError_t launch_conv_generic(const ConvLayer &L, const ConvProblem &P, const EpiParams &E, cudaStream_t st)
{
    dim3 grid((P.H * P.W + GM - 1) / GM, (L.n + GN - 1) / GN, P.n_img);
    conv_generic_kernel<<<grid, 256, 0, st>>>(P.in, L.w, L.bias, P.n_img, P.H, P.W, L.c_in, L.n, L.n_pad, L.taps, L.groups, E);
    return cudaGetLastError();
}

// ---- A6: depthwise 3x3, zero pad, bias.  HBM-bound: each thread owns 8 channels (one 16-byte
// vector) of a run of DW_X horizontally adjacent pixels and slides a 3-column register window, so every input
// vector is loaded 3 times (once per output row it feeds; the row neighbours hit L1/L2), and stored once.
constexpr int DW_X = 4;

__global__ void __launch_bounds__(256) dwconv3x3_kernel(const bf16 *__restrict__ in, bf16 *__restrict__ out,
                                                        const float *__restrict__ w9c, const float *__restrict__ bias,
                                                        int n_img, int H, int W, int C)
{
    const int cv = C / 8;                               // channel vectors per pixel
    const int xr = (W + DW_X - 1) / DW_X;               // pixel runs per row
    const long long total = (long long)n_img * H * xr * cv;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int c8 = int(t % cv);
        long long r = t / cv;
        const int xrun = int(r % xr); r /= xr;
        const int y = int(r % H);
        const int img = int(r / H);
        const int c0 = c8 * 8, x0 = xrun * DW_X;
        float wv[9][8], bv[8];
#pragma unroll
        for (int k = 0; k < 9; ++k) {
            const float4 lo = *reinterpret_cast<const float4 *>(w9c + k * C + c0);
            const float4 hi = *reinterpret_cast<const float4 *>(w9c + k * C + c0 + 4);
            wv[k][0] = lo.x; wv[k][1] = lo.y; wv[k][2] = lo.z; wv[k][3] = lo.w;
            wv[k][4] = hi.x; wv[k][5] = hi.y; wv[k][6] = hi.z; wv[k][7] = hi.w;
        }
        {
            const float4 lo = *reinterpret_cast<const float4 *>(bias + c0), hi = *reinterpret_cast<const float4 *>(bias + c0 + 4);
            bv[0] = lo.x; bv[1] = lo.y; bv[2] = lo.z; bv[3] = lo.w; bv[4] = hi.x; bv[5] = hi.y; bv[6] = hi.z; bv[7] = hi.w;
        }
        const bf16 *img_in = in + (long long)img * H * W * C;
        float acc[DW_X][8];
#pragma unroll
        for (int i = 0; i < DW_X; ++i)
#pragma unroll
            for (int e = 0; e < 8; ++e) acc[i][e] = bv[e];
#pragma unroll
        for (int dy = 0; dy < 3; ++dy) {
            const int yy = y + dy - 1;
            if (yy < 0 || yy >= H) continue;
#pragma unroll
            for (int xi = 0; xi < DW_X + 2; ++xi) {     // input column x0 - 1 + xi feeds outputs xi-2 .. xi
                const int xx = x0 - 1 + xi;
                if (xx < 0 || xx >= W) continue;
                const uint4 v = *reinterpret_cast<const uint4 *>(img_in + ((long long)yy * W + xx) * C + c0);
                const bf16 *ve = reinterpret_cast<const bf16 *>(&v);
                float f[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) f[e] = __bfloat162float(ve[e]);
#pragma unroll
                for (int dx = 0; dx < 3; ++dx) {
                    const int oi = xi - dx;             // output index whose tap dx reads this column
                    if (oi < 0 || oi >= DW_X) continue;
#pragma unroll
                    for (int e = 0; e < 8; ++e) acc[oi][e] = fmaf(wv[dy * 3 + dx][e], f[e], acc[oi][e]);
                }
            }
        }
#pragma unroll
        for (int i = 0; i < DW_X; ++i) {
            if (x0 + i >= W) continue;
            uint4 o;
            bf16 *oe = reinterpret_cast<bf16 *>(&o);
#pragma unroll
            for (int e = 0; e < 8; ++e) oe[e] = __float2bfloat16_rn(acc[i][e]);
            *reinterpret_cast<uint4 *>(out + (((long long)img * H + y) * W + x0 + i) * C + c0) = o;
        }
    }
}

cudaError_t launch_dwconv3x3(const bf16 *in, bf16 *out, const float *w9c, const float *bias, int n_img, int H, int W,
                             int C, cudaStream_t st)
{
    const long long total = (long long)n_img * H * ((W + DW_X - 1) / DW_X) * (C / 8);
    long long blocks = (total + 255) / 256;
    if (blocks > 148LL * 64) blocks = 148LL * 64;
    dwconv3x3_kernel<<<(unsigned)blocks, 256, 0, st>>>(in, out, w9c, bias, n_img, H, W, C);
    return cudaGetLastError();
}

}  // namespace ufnvc
