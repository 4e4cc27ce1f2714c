// GPU rANS ENCODE of the residual r ("GPU rANS encode with the mirrored warp scan"), the exact
// mirror of the A3 decoder (rans.cu) and of the oracle's O4 encoder: same container, byte for byte.
// "the result r_i is arithmetically encoded using scale sigma_i" -- the tables depend on the scale only.
//
// One block per substream, one warp per warp-stream (32 interleaved 32-bit states, 16-bit words, 16-bit probabilities).
// The encoder walks the steps DOWN; inside a step the lanes emit in DESCENDING lane order (the decoder pulls words in
// ascending lane order), so lane l's word lands at  n_words_so_far + popc(ballot above l)  -- the mirrored warp scan --
// in a scratch run that is written out reversed at the end.  Container of a substream:
//   u32 hdr[2G] = {byte offset of warp-stream g, n_words_g};  per g: u32 state[32], u16 word[n_words_g], 4-byte padded.
// A second kernel packs the substreams back to back and writes the offset table.
#include "tc_ptx.cuh"
#include "ufnvc_internal.h"

namespace ufnvc {

// A substream is coded by a CLUSTER of `ranks` blocks of blockDim.x / 32 warp-streams each (ranks = 1: one block): with all 16
// warp-streams of a 1080p substream on one SM the kernel was bound by that SM's issue slots (16 warps x ~150 instructions per
// step).  The blocks only meet at the end, to lay the warp-streams out one behind the other: their byte counts travel through
// distributed shared memory.
__global__ void __launch_bounds__(512) rans_encode_kernel(RansEncParams p, int ranks)
{
    __shared__ uint32_t s_bytes[32];                                   // bytes of warp-stream g (states + words, padded), all ranks
    const int sub = blockIdx.x / ranks;                                 // chunk * n_sub + s
    const int rank = ranks > 1 ? int(cluster_ctarank()) : 0;
    const int chunk = sub / p.n_sub, s = sub % p.n_sub;
    const int g = rank * int(blockDim.x >> 5) + int(threadIdx.x >> 5), lane = threadIdx.x & 31;
    const int G = p.W >> 5;
    const int row0 = s * p.rows_per_sub;
    const int rows = min(p.rows_per_sub, p.h - row0);
    const int n = rows * p.w * p.c_y;
    const long long ebase = ((long long)chunk * p.h + row0) * p.w * p.c_y;   // stream order == channels-last order
    const int n_steps = (n + p.W - 1) / p.W;
    uint16_t *tmp = p.tmp_words + ((size_t)sub * G + g) * p.tmp_stride;      // this warp-stream's scratch run
    uint8_t *out = p.stage + (size_t)sub * p.stage_stride;

    uint32_t x = 1u << 16, nw = 0, bad = 0;
    // The symbol, its index and the table entry of a step do not depend on the coder state: they are fetched for kB steps at a
    // time (two rounds of independent loads), so the serial chain of a step holds no memory latency -- a load -> load -> load
    // chain inside every step had made the kernel 120 x 0.95 us per 1080p substream.
    constexpr int kB = 16;
    for (int j0 = n_steps - 1; j0 >= 0; j0 -= kB) {
        uint32_t cf[kB];                                               // c | freq << 16; 0 = no symbol here; 0xFFFFFFFF = malformed input
        {
            int pos[kB];
            uint32_t k[kB];
#pragma unroll
            for (int t = 0; t < kB; ++t) {
                const int i = (j0 - t) * p.W + g * 32 + lane;
                const bool valid = j0 - t >= 0 && i < n;
                pos[t] = valid ? int(__ldg(p.sym + ebase + i)) + 127 : -1000;
                k[t] = valid ? uint32_t(__ldg(p.idx + ebase + i)) : 0u;
            }
#pragma unroll
            for (int t = 0; t < kB; ++t) {
                if (pos[t] == -1000) cf[t] = 0u;
                else if (pos[t] < 0 || pos[t] > 254 || k[t] >= uint32_t(p.n_buckets)) cf[t] = 0xFFFFFFFFu;
                else cf[t] = __ldg(p.cf + k[t] * 256 + pos[t]);             // freq >= 1: never 0, and freq <= 65282: never 0xFFFFFFFF
            }
        }
#pragma unroll
        for (int t = 0; t < kB; ++t) {
            if (j0 - t < 0) break;                                     // (warp-uniform)
            if (cf[t] == 0xFFFFFFFFu) bad = 1;
            const bool live = cf[t] != 0u && !bad;
            const uint32_t f = live ? cf[t] >> 16 : 1u, cs = cf[t] & 0xFFFFu;
            const bool emit = live && (uint64_t(x) >= (uint64_t(f) << 16));
            const uint32_t m = __ballot_sync(0xFFFFFFFFu, emit);
            if (emit) {
                tmp[nw + __popc(m >> 1 >> lane)] = uint16_t(x & 0xFFFFu);   // lanes above this one emit first
                x >>= 16;
            }
            nw += __popc(m);
            if (live) x = ((x / f) << 16) + (x % f) + cs;
        }
    }
    if (__any_sync(0xFFFFFFFFu, bad) && lane == 0) atomicOr(p.status, UFNVC_STREAM_BAD_HEADER);

    // ---- layout of the substream: header, then the warp-streams in order ----
    if (ranks == 1) {
        if (lane == 0) s_bytes[g] = (128u + 2u * nw + 3u) & ~3u;
        __syncthreads();
    } else {
        if (lane < ranks) {                                             // lane r tells block r of the cluster
            const uint32_t remote = mapa_rank(smem_u32(&s_bytes[g]), uint32_t(lane));
            asm volatile("st.shared::cluster.u32 [%0], %1;" ::"r"(remote), "r"((128u + 2u * nw + 3u) & ~3u) : "memory");
        }
        cluster_sync_all();                                             // (release / acquire at cluster scope)
    }
    uint32_t pos = 8u * G;
    for (int q = 0; q < g; ++q) pos += s_bytes[q];
    if (lane == 0) {
        reinterpret_cast<uint32_t *>(out)[2 * g] = pos;
        reinterpret_cast<uint32_t *>(out)[2 * g + 1] = nw;
    }
    reinterpret_cast<uint32_t *>(out + pos)[lane] = x;
    uint16_t *wout = reinterpret_cast<uint16_t *>(out + pos + 128);
    __syncwarp();                                                       // scratch words written by other lanes
    for (uint32_t q0 = 0; q0 < nw; q0 += 32 * 8) {                     // eight independent loads in flight per lane (one at a time was
        uint16_t v[8];                                                  // 120 L2 round trips per warp-stream: most of the kernel)
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const uint32_t q = q0 + uint32_t(u) * 32 + lane;
            v[u] = q < nw ? tmp[nw - 1 - q] : uint16_t(0);
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const uint32_t q = q0 + uint32_t(u) * 32 + lane;
            if (q < nw) wout[q] = v[u];
        }
    }
    if ((nw & 1u) && lane == 0) wout[nw] = 0;                           // zero padding to 4 bytes
    if (threadIdx.x == 0 && rank == 0) {
        uint32_t total = 8u * G;
        for (int q = 0; q < G; ++q) total += s_bytes[q];
        p.sizes[sub] = total;
    }
}

// pack: offsets = exclusive scan of the substream sizes; every substream is copied to its place (sizes are multiples of 4).
// One block per (substream, part): each block sums the sizes before its substream and the total itself (a few hundred words),
// so no block waits for another; a single-block version of this copy took longer than the encode.
constexpr int kPackParts = 4;
__global__ void __launch_bounds__(256) rans_pack_kernel(RansEncParams p, int n_total_sub)
{
    __shared__ uint32_t s_before, s_total;
    const int sub = blockIdx.x / kPackParts, part = blockIdx.x % kPackParts;
    if (threadIdx.x < 32) {
        uint32_t before = 0, total = 0;
        for (int i = threadIdx.x; i < n_total_sub; i += 32) {
            const uint32_t sz = p.sizes[i];
            total += sz;
            if (i < sub) before += sz;
        }
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1) {
            before += __shfl_xor_sync(0xFFFFFFFFu, before, d);
            total += __shfl_xor_sync(0xFFFFFFFFu, total, d);
        }
        if (threadIdx.x == 0) { s_before = before; s_total = total; }
    }
    __syncthreads();
    const uint32_t o0 = s_before, total = s_total;
    if (part == 0 && threadIdx.x == 0) {
        p.sub_off[sub] = o0;
        if (sub == n_total_sub - 1) {
            p.sub_off[n_total_sub] = total;
            if ((size_t)total > p.cap) atomicOr(p.status, UFNVC_STREAM_BAD_WORD_COUNT);   // output buffer too small: offsets only
        }
    }
    if ((size_t)total > p.cap) return;
    const uint32_t *src = reinterpret_cast<const uint32_t *>(p.stage + (size_t)sub * p.stage_stride);
    uint32_t *dst = reinterpret_cast<uint32_t *>(p.bits_out + o0);
    const uint32_t words = p.sizes[sub] >> 2;
    const uint32_t stride = kPackParts * blockDim.x;
    for (uint32_t q0 = uint32_t(part) * blockDim.x + threadIdx.x; q0 < words; q0 += 4 * stride) {
        uint32_t v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = q0 + u * stride < words ? src[q0 + u * stride] : 0u;
#pragma unroll
        for (int u = 0; u < 4; ++u) if (q0 + u * stride < words) dst[q0 + u * stride] = v[u];
    }
}

cudaError_t launch_rans_encode(const RansEncParams &p, LaunchStream st)
{
    const int n_total = p.n_chunks * p.n_sub;
    const int G = p.W / 32;
    const int ranks = (G % 4 == 0 && G / 4 <= 8 && G > 4) ? G / 4 : 1;           // 4 warp-streams per block where that splits a substream evenly
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(unsigned(n_total * ranks)); cfg.blockDim = dim3(unsigned(p.W / ranks)); cfg.dynamicSmemBytes = 0; cfg.stream = st.s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = unsigned(ranks); attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = ranks > 1 ? 1u : 0u;
    cudaError_t e = cudaLaunchKernelEx(&cfg, rans_encode_kernel, p, ranks);
    if (e != cudaSuccess) return e;
    rans_pack_kernel<<<n_total * kPackParts, 256, 0, st>>>(p, n_total);
    return cudaGetLastError();
}

}  // namespace ufnvc
