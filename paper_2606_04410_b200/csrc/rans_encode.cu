// GPU rANS ENCODE of the residual r ("GPU rANS encode with the mirrored warp scan"), the exact
// mirror of the A3 decoder (rans.cu) and of the oracle's O4 encoder: same container, byte for byte.
// "the result r_i is arithmetically encoded using scale sigma_i" -- the tables depend on the scale only.
//
// One block per substream, one warp per warp-stream (32 interleaved 32-bit states, 16-bit words, 16-bit probabilities).
// The encoder walks the steps DOWN; inside a step the lanes emit in DESCENDING lane order (the decoder pulls words in
// ascending lane order), so lane l's word lands at  n_words_so_far + popc(ballot above l)  -- the mirrored warp scan --
// in a scratch run that is written out reversed at the end.  Container of a substream:
//   u32 hdr[2G] = {byte offset of warp-stream g, n_words_g};  per g: u32 state[32], u16 word[n_words_g], 4-byte padded.
// A second, single-block kernel packs the substreams back to back and writes the offset table.
#include "ufnvc_internal.h"

namespace ufnvc {

__global__ void __launch_bounds__(512) rans_encode_kernel(RansEncParams p)
{
    __shared__ uint32_t s_bytes[16];                                   // bytes of warp-stream g (states + words, padded)
    const int sub = blockIdx.x;                                         // chunk * n_sub + s
    const int chunk = sub / p.n_sub, s = sub % p.n_sub;
    const int g = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int G = p.W >> 5;
    const int row0 = s * p.rows_per_sub;
    const int rows = min(p.rows_per_sub, p.h - row0);
    const int n = rows * p.w * p.c_y;
    const long long ebase = ((long long)chunk * p.h + row0) * p.w * p.c_y;   // stream order == channels-last order
    const int n_steps = (n + p.W - 1) / p.W;
    uint16_t *tmp = p.tmp_words + ((size_t)sub * G + g) * p.tmp_stride;      // this warp-stream's scratch run
    uint8_t *out = p.stage + (size_t)sub * p.stage_stride;

    uint32_t x = 1u << 16, nw = 0, bad = 0;
    for (int j = n_steps - 1; j >= 0; --j) {
        const int i = j * p.W + g * 32 + lane;
        const bool valid = i < n;
        uint32_t f = 1, cs = 0;
        if (valid) {
            const int pos = int(p.sym[ebase + i]) + 127;
            const uint32_t k = p.idx[ebase + i];
            if (pos < 0 || pos > 254 || k >= uint32_t(p.n_buckets)) bad = 1;
            else {
                const uint32_t cf = p.cf[k * 256 + pos];
                cs = cf & 0xFFFFu; f = cf >> 16;
            }
        }
        const bool emit = valid && !bad && (uint64_t(x) >= (uint64_t(f) << 16));
        const uint32_t m = __ballot_sync(0xFFFFFFFFu, emit);
        if (emit) {
            tmp[nw + __popc(m >> 1 >> lane)] = uint16_t(x & 0xFFFFu);   // lanes above this one emit first
            x >>= 16;
        }
        nw += __popc(m);
        if (valid && !bad) x = ((x / f) << 16) + (x % f) + cs;
    }
    if (__any_sync(0xFFFFFFFFu, bad) && lane == 0) atomicOr(p.status, UFNVC_STREAM_BAD_HEADER);

    // ---- layout of the substream: header, then the warp-streams in order ----
    if (lane == 0) s_bytes[g] = (128u + 2u * nw + 3u) & ~3u;
    __syncthreads();
    uint32_t pos = 8u * G;
    for (int q = 0; q < g; ++q) pos += s_bytes[q];
    if (lane == 0) {
        reinterpret_cast<uint32_t *>(out)[2 * g] = pos;
        reinterpret_cast<uint32_t *>(out)[2 * g + 1] = nw;
    }
    reinterpret_cast<uint32_t *>(out + pos)[lane] = x;
    uint16_t *wout = reinterpret_cast<uint16_t *>(out + pos + 128);
    __syncwarp();                                                       // scratch words written by other lanes
    for (uint32_t q = lane; q < nw; q += 32) wout[q] = tmp[nw - 1 - q];
    if ((nw & 1u) && lane == 0) wout[nw] = 0;                           // zero padding to 4 bytes
    if (threadIdx.x == 0) {
        uint32_t total = 8u * G;
        for (int q = 0; q < G; ++q) total += s_bytes[q];
        p.sizes[sub] = total;
    }
}

// pack: offsets = exclusive scan of the substream sizes; copy every substream to its place (sizes are multiples of 4)
__global__ void __launch_bounds__(1024) rans_pack_kernel(RansEncParams p, int n_total_sub)
{
    extern __shared__ uint32_t s_off[];                                 // n_total_sub + 1
    if (threadIdx.x == 0) {
        uint32_t o = 0;
        for (int i = 0; i < n_total_sub; ++i) { s_off[i] = o; o += p.sizes[i]; }
        s_off[n_total_sub] = o;
        if ((size_t)o > p.cap) atomicOr(p.status, UFNVC_STREAM_BAD_WORD_COUNT);    // output buffer too small: nothing is copied
    }
    __syncthreads();
    for (int i = threadIdx.x; i <= n_total_sub; i += blockDim.x) p.sub_off[i] = s_off[i];
    if ((size_t)s_off[n_total_sub] > p.cap) return;
    for (int sub = 0; sub < n_total_sub; ++sub) {
        const uint32_t *src = reinterpret_cast<const uint32_t *>(p.stage + (size_t)sub * p.stage_stride);
        uint32_t *dst = reinterpret_cast<uint32_t *>(p.bits_out + s_off[sub]);
        const uint32_t words = (s_off[sub + 1] - s_off[sub]) >> 2;
        for (uint32_t q = threadIdx.x; q < words; q += blockDim.x) dst[q] = src[q];
    }
}

cudaError_t launch_rans_encode(const RansEncParams &p, LaunchStream st)
{
    const int n_total = p.n_chunks * p.n_sub;
    rans_encode_kernel<<<n_total, p.W, 0, st>>>(p);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    rans_pack_kernel<<<1, 1024, (n_total + 1) * sizeof(uint32_t), st>>>(p, n_total);
    return cudaGetLastError();
}

}  // namespace ufnvc
