// NEXT-4 (R24): the encode side that feeds the GPU rANS encoder, and the colour interface.
// "transforming it to 1/8 resolution via patch embedding ... fed into a chunk encoder"; "After
// quantization via r = round(y - mu), the result r is arithmetically encoded using scale sigma"; PAPER.md:384 (Supp. C): a
// unified YUV444 interface, BT.709 for RGB.  The dense layers of the encoder (patch embedding, fold over frames, DC blocks,
// latent head) run on the decoder's tcgen05 conv and fused-MLP kernels (decode.cu strings them together); this file holds the
// small kernels around them: the 8x8 patch gather, the hyper-encoder, the quantiser and the colour conversions.
#include "ufnvc_internal.h"

namespace ufnvc {

// ---- E1 gather: frames fp32 planar [n_img][3][height][width] -> bf16 NHWC [n_img][H/8][W/8][192], channel (8 i + j) 3 + c =
// pixel (8 y + i, 8 x + j) of plane c; rows / columns past (height, width) are the codec's zero padding (R16).  A thread owns
// one patch row i of one 1/8-resolution pixel: three 32-byte reads (whole sectors), one 48-byte write; the 8 threads of a
// pixel write its 384 bytes contiguously.
__global__ void __launch_bounds__(256) enc_patchify_kernel(const float *__restrict__ frames, bf16 *__restrict__ out, int n_img, int height,
                                                           int width, int H8, int W8)
{
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const long long total = (long long)n_img * H8 * W8 * 8;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int i = int(t & 7);
        long long pix = t >> 3;
        const int x8 = int(pix % W8); pix /= W8;
        const int y8 = int(pix % H8);
        const int img = int(pix / H8);
        const int yy = 8 * y8 + i, x0 = 8 * x8;
        float v[3][8];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const float *src = frames + (((long long)img * 3 + c) * height + yy) * width + x0;
            if (yy < height && x0 + 8 <= width && (reinterpret_cast<uintptr_t>(src) & 15) == 0) {
                const float4 a = *reinterpret_cast<const float4 *>(src), b = *reinterpret_cast<const float4 *>(src + 4);
                v[c][0] = a.x; v[c][1] = a.y; v[c][2] = a.z; v[c][3] = a.w; v[c][4] = b.x; v[c][5] = b.y; v[c][6] = b.z; v[c][7] = b.w;
            } else {
#pragma unroll
                for (int j = 0; j < 8; ++j) v[c][j] = (yy < height && x0 + j < width) ? src[j] : 0.0f;
            }
        }
        __nv_bfloat162 o[12];                                       // channels (8 i + j) 3 + c, j = 0..7, c = 0..2: 24 consecutive
        float f[24];
#pragma unroll
        for (int j = 0; j < 8; ++j)
#pragma unroll
            for (int c = 0; c < 3; ++c) f[j * 3 + c] = v[c][j];
#pragma unroll
        for (int e = 0; e < 12; ++e) o[e] = __floats2bfloat162_rn(f[2 * e], f[2 * e + 1]);
        uint4 *dst = reinterpret_cast<uint4 *>(out + (((long long)img * H8 + y8) * W8 + x8) * 192 + i * 24);
        const uint4 *os = reinterpret_cast<const uint4 *>(o);
        dst[0] = os[0]; dst[1] = os[1]; dst[2] = os[2];
    }
}

cudaError_t launch_enc_patchify(const float *frames, bf16 *out, int n_img, int height, int width, int H8, int W8, LaunchStream st)
{
    const long long total = (long long)n_img * H8 * W8 * 8;
    long long blocks = (total + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    return launch_pdl(enc_patchify_kernel, unsigned(blocks), 256u, 0, st, 1, frames, out, n_img, height, width, H8, W8);
}

// ---- E6 hyper-encoder, fp32 on CUDA cores (0.35 GMAC per 1080p chunk).  Layer 0: a = ReLU(W0 Y4 + b0), Y4 = space-to-depth x4
// of y (zero past the latent's edge), K = 16 c_y with k = (4 i + j) c_y + c.  A block is 8 z-pixels x 64 outputs x 8 slices of K:
// the 8 input vectors sit in shared memory, thread (o, slice) walks its K / 8 with coalesced weight reads w0[k][o], eight loads in
// flight per thread; the slices are summed in a fixed order through shared memory.  (A first version walked all of K in one thread
// with one load per step: 313 us of L2 latency for 0.27 GMAC.)
constexpr int kHencPix = 8, kHencO = 64, kHencSlices = 8;
__global__ void __launch_bounds__(kHencO * kHencSlices) henc0_kernel(const float *__restrict__ y, const float *__restrict__ w0,
                                                                     const float *__restrict__ b0, float *__restrict__ a, int n_img, int h, int w,
                                                                     int hz, int wz, int c_y, int c_h)
{
    extern __shared__ float xin[];                                  // [kHencPix][16 c_y], then the slice sums [kHencSlices][kHencPix][kHencO]
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int K = 16 * c_y, M = n_img * hz * wz, m0 = blockIdx.x * kHencPix;
    float *red = xin + kHencPix * K;
    // one warp per (z-pixel, sub-pixel) segment of c_y contiguous floats: the address arithmetic is per segment, not per element
    for (int seg = threadIdx.x >> 5; seg < kHencPix * 16; seg += blockDim.x >> 5) {
        const int pi = seg >> 4, ij = seg & 15, m = m0 + pi;
        const float *src = nullptr;
        if (m < M) {
            const int img = m / (hz * wz), r = m % (hz * wz), zy = r / wz, zx = r % wz;
            const int ly = 4 * zy + (ij >> 2), lx = 4 * zx + (ij & 3);
            if (ly < h && lx < w) src = y + (((long long)img * h + ly) * w + lx) * c_y;
        }
        float *dst = xin + pi * K + ij * c_y;
        for (int c = threadIdx.x & 31; c < c_y; c += 32) dst[c] = src ? src[c] : 0.0f;
    }
    __syncthreads();
    const int ol = threadIdx.x % kHencO, ks = threadIdx.x / kHencO, o = blockIdx.y * kHencO + ol;
    const int kn = K / kHencSlices, k0 = ks * kn;                   // (K is a multiple of 128)
    float acc[kHencPix];
#pragma unroll
    for (int pi = 0; pi < kHencPix; ++pi) acc[pi] = 0.0f;
    if (o < c_h) {
        const float *wp = w0 + (long long)k0 * c_h + o;
        for (int k = 0; k < kn; k += 8) {
            float wv[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) wv[u] = __ldg(wp + (long long)(k + u) * c_h);
#pragma unroll
            for (int pi = 0; pi < kHencPix; ++pi) {                 // (warp-uniform addresses: broadcast 128-bit loads)
                const float4 x0 = *reinterpret_cast<const float4 *>(xin + pi * K + k0 + k), x1 = *reinterpret_cast<const float4 *>(xin + pi * K + k0 + k + 4);
                acc[pi] = fmaf(wv[0], x0.x, acc[pi]); acc[pi] = fmaf(wv[1], x0.y, acc[pi]); acc[pi] = fmaf(wv[2], x0.z, acc[pi]); acc[pi] = fmaf(wv[3], x0.w, acc[pi]);
                acc[pi] = fmaf(wv[4], x1.x, acc[pi]); acc[pi] = fmaf(wv[5], x1.y, acc[pi]); acc[pi] = fmaf(wv[6], x1.z, acc[pi]); acc[pi] = fmaf(wv[7], x1.w, acc[pi]);
            }
        }
    }
#pragma unroll
    for (int pi = 0; pi < kHencPix; ++pi) red[(ks * kHencPix + pi) * kHencO + ol] = acc[pi];
    __syncthreads();
    {
        const int pi = threadIdx.x / kHencO;                        // 8 pixels x 64 outputs = one result per thread
        float v = 0.0f;
#pragma unroll
        for (int q = 0; q < kHencSlices; ++q) v += red[(q * kHencPix + pi) * kHencO + ol];
        if (o < c_h && m0 + pi < M) a[(long long)(m0 + pi) * c_h + o] = fmaxf(v + b0[o], 0.0f);
    }
}

// Layer 1: zf = conv3x3(a; c_h -> c_z), z = clip(rint(zf), -127, 127) as int16, planar [n][c_z][pz] (what A1 reads).
// A block is 4 z-pixels x 64 outputs x 8 slices of K = 9 c_h, same scheme.
constexpr int kHenc1Pix = 4;
__global__ void __launch_bounds__(kHencO * kHencSlices) henc1_kernel(const float *__restrict__ a, const float *__restrict__ w1,
                                                                     const float *__restrict__ b1, int16_t *__restrict__ z, float *__restrict__ zf_tap,
                                                                     int n_img, int hz, int wz, int c_h, int c_z)
{
    extern __shared__ float ain[];                                  // [kHenc1Pix][9][c_h], then [kHencSlices][kHenc1Pix][kHencO]
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int pz = hz * wz, M = n_img * pz, K = 9 * c_h, m0 = blockIdx.x * kHenc1Pix;
    float *red = ain + kHenc1Pix * K;
    for (int e = threadIdx.x; e < kHenc1Pix * K; e += blockDim.x) {
        const int pi = e / K, k = e - pi * K, m = m0 + pi;
        float v = 0.0f;
        if (m < M) {
            const int img = m / pz, r = m % pz, zy = r / wz, zx = r % wz;
            const int tap = k / c_h, c = k - tap * c_h, yy = zy + tap / 3 - 1, xx = zx + tap % 3 - 1;
            if (yy >= 0 && yy < hz && xx >= 0 && xx < wz) v = a[(((long long)img * hz + yy) * wz + xx) * c_h + c];
        }
        ain[e] = v;
    }
    __syncthreads();
    const int ol = threadIdx.x % kHencO, ks = threadIdx.x / kHencO, o = blockIdx.y * kHencO + ol;
    const int kn = K / kHencSlices, k0 = ks * kn;                   // (c_h is a multiple of 16: kn is a multiple of 8)
    float acc[kHenc1Pix];
#pragma unroll
    for (int pi = 0; pi < kHenc1Pix; ++pi) acc[pi] = 0.0f;
    if (o < c_z) {
        const float *wp = w1 + (long long)k0 * c_z + o;           // w1[tap][c][o]
        for (int k = 0; k < kn; k += 8) {
            float wv[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) wv[u] = __ldg(wp + (long long)(k + u) * c_z);
#pragma unroll
            for (int u = 0; u < 8; ++u)
#pragma unroll
                for (int pi = 0; pi < kHenc1Pix; ++pi) acc[pi] = fmaf(wv[u], ain[pi * K + k0 + k + u], acc[pi]);
        }
    }
#pragma unroll
    for (int pi = 0; pi < kHenc1Pix; ++pi) red[(ks * kHenc1Pix + pi) * kHencO + ol] = acc[pi];
    __syncthreads();
    if (threadIdx.x < kHenc1Pix * kHencO) {
        const int pi = threadIdx.x / kHencO, m = m0 + pi;
        float v = 0.0f;
#pragma unroll
        for (int q = 0; q < kHencSlices; ++q) v += red[(q * kHenc1Pix + pi) * kHencO + ol];
        if (o < c_z && m < M) {
            v += b1[o];
            const int img = m / pz, r = m % pz;
            const float qv = fminf(fmaxf(rintf(v), -127.0f), 127.0f);
            z[((long long)img * c_z + o) * pz + r] = int16_t(qv);
            if (zf_tap) zf_tap[((long long)img * c_z + o) * pz + r] = v;
        }
    }
}

cudaError_t launch_hyper_encoder(const float *y, const float *w0, const float *b0, const float *w1, const float *b1, float *a, int16_t *z,
                                 float *zf_tap, int n_img, int h, int w, int hz, int wz, int c_y, int c_h, int c_z, LaunchStream st)
{
    const int M = n_img * hz * wz;
    const size_t smem0 = (size_t(kHencPix) * 16 * c_y + size_t(kHencSlices) * kHencPix * kHencO) * sizeof(float);
    const size_t smem1 = (size_t(kHenc1Pix) * 9 * c_h + size_t(kHencSlices) * kHenc1Pix * kHencO) * sizeof(float);
    if (smem0 > 200 * 1024 || smem1 > 200 * 1024 || (16 * c_y) % (8 * kHencSlices) || (9 * c_h) % (8 * kHencSlices)) return cudaErrorInvalidValue;
    cudaError_t e = cudaFuncSetAttribute(henc0_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem0));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(henc1_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem1));
    if (e != cudaSuccess) return e;
    const dim3 g0(unsigned((M + kHencPix - 1) / kHencPix), unsigned((c_h + kHencO - 1) / kHencO));
    const dim3 g1(unsigned((M + kHenc1Pix - 1) / kHenc1Pix), unsigned((c_z + kHencO - 1) / kHencO));
    e = launch_pdl_grid_smem(henc0_kernel, g0, kHencO * kHencSlices, smem0, st, y, w0, b0, a, n_img, h, w, hz, wz, c_y, c_h);
    if (e != cudaSuccess) return e;
    return launch_pdl_grid_smem(henc1_kernel, g1, kHencO * kHencSlices, smem1, st, a, w1, b1, z, zf_tap, n_img, hz, wz, c_h, c_z);
}

// ---- E8 quantiser: r = clip(rint(y - mu), -127, 127), round half to even, in fp32.
__global__ void __launch_bounds__(256) enc_quantise_kernel(const float *__restrict__ y, const float *__restrict__ mu, int16_t *__restrict__ sym,
                                                           long long n)
{
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    for (long long i = (blockIdx.x * (long long)blockDim.x + threadIdx.x) * 4; i < n; i += (long long)gridDim.x * blockDim.x * 4) {
        if (i + 4 <= n) {
            const float4 a = *reinterpret_cast<const float4 *>(y + i), b = *reinterpret_cast<const float4 *>(mu + i);
            short4 r;
            r.x = short(fminf(fmaxf(rintf(a.x - b.x), -127.0f), 127.0f)); r.y = short(fminf(fmaxf(rintf(a.y - b.y), -127.0f), 127.0f));
            r.z = short(fminf(fmaxf(rintf(a.z - b.z), -127.0f), 127.0f)); r.w = short(fminf(fmaxf(rintf(a.w - b.w), -127.0f), 127.0f));
            *reinterpret_cast<short4 *>(sym + i) = r;
        } else {
            for (long long j = i; j < n; ++j) sym[j] = int16_t(fminf(fmaxf(rintf(y[j] - mu[j]), -127.0f), 127.0f));
        }
    }
}

cudaError_t launch_enc_quantise(const float *y, const float *mu, int16_t *sym, long long n, LaunchStream st)
{
    long long blocks = (n / 4 + 255) / 256 + 1;
    if (blocks > 148 * 8) blocks = 148 * 8;
    return launch_pdl(enc_quantise_kernel, unsigned(blocks), 256u, 0, st, 1, y, mu, sym, n);
}

// ---- colour interface: full-range BT.709 on [0,1] floats, planar [n][3][H][W] in and out.
__global__ void __launch_bounds__(256) colour_kernel(const float *__restrict__ in, float *__restrict__ out, long long plane, long long n_img, int to_yuv)
{
    const long long total = plane * n_img;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const long long img = t / plane, p = t - img * plane;
        const float *s = in + img * 3 * plane + p;
        float *d = out + img * 3 * plane + p;
        const float a = s[0], b = s[plane], c = s[2 * plane];
        if (to_yuv) {
            const float yy = 0.2126f * a + 0.7152f * b + 0.0722f * c;
            d[0] = yy; d[plane] = (c - yy) / 1.8556f + 0.5f; d[2 * plane] = (a - yy) / 1.5748f + 0.5f;
        } else {
            const float r = a + 1.5748f * (c - 0.5f), bl = a + 1.8556f * (b - 0.5f);
            d[0] = r; d[plane] = (a - 0.2126f * r - 0.0722f * bl) / 0.7152f; d[2 * plane] = bl;
        }
    }
}

cudaError_t launch_colour(const float *in, float *out, long long plane, long long n_img, bool to_yuv, cudaStream_t st)
{
    long long blocks = (plane * n_img + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    if (blocks < 1) blocks = 1;
    colour_kernel<<<unsigned(blocks), 256, 0, st>>>(in, out, plane, n_img, to_yuv ? 1 : 0);
    return cudaGetLastError();
}

}  // namespace ufnvc
