// ufnvc_encode_chunk_dev_static: the GPU rANS encoder (rans_encode.cu) for callers that may
// not allocate device memory -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
// ufnvc_encode_chunk_dev allocates its scratch (the per-warp-stream word runs the encoder writes in reverse, the staged
// substreams and their sizes) with cudaMalloc on its first call; this entry point runs the SAME kernels with that scratch in a
// file-scope __device__ array of fixed size, so the call itself allocates nothing.
//
// The array's name is a host-side stand-in in host code, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, taken once per handle at ufnvc_create with the handle's device current (static_scratch_address below;
// the handle keeps it, so two handles on two GPUs each hold the address valid on their own device).
//
// Every GPU that loads the library holds the array until the process exits.  Every call, on every handle of a device, shares
// it, and it keeps the previous call's contents: the encoder writes every byte it later reads (word runs, headers, states,
// padding), the per-substream size table is cleared on the stream before the kernels run, and two calls that overlap on the
// GPU (different streams, no ordering between them) race on it -- callers serialise them.
#include "handle.h"

namespace {

constexpr size_t kStaticScratchBytes = size_t(UFNVC_STATIC_SCRATCH_BYTES);
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

inline size_t align256(size_t v) { return (v + 255) & ~size_t(255); }

}  // namespace

namespace ufnvc {

// Device address of the static scratch on the CURRENT device (set-up time, not under stream capture).
cudaError_t static_scratch_address(void **ptr)
{
    *ptr = nullptr;
    return cudaGetSymbolAddress(ptr, g_static_scratch);
}

}  // namespace ufnvc

extern "C" int ufnvc_encode_chunk_dev_static(ufnvc_handle *h, int n_chunks, const uint8_t *idx_dev, const int16_t *sym_dev,
                                             uint8_t *bits_dev, size_t cap, uint32_t *sub_off_dev, void *cuda_stream)
{
    using namespace ufnvc;
    if (!h) return UFNVC_E_INVALID_ARG;
    if (n_chunks < 1 || n_chunks > h->max_chunks) return fail(h, UFNVC_E_INVALID_ARG, "n_chunks outside [1, max_chunks_per_call]");
    if (!idx_dev || !sym_dev || !bits_dev || !sub_off_dev) return fail(h, UFNVC_E_INVALID_ARG, "null device pointer");
    if (reinterpret_cast<uintptr_t>(bits_dev) & 3) return fail(h, UFNVC_E_INVALID_ARG, "bits_dev must be 4-byte aligned");
    if (!h->static_scratch) return fail(h, UFNVC_E_CUDA, "static scratch unavailable: cudaGetSymbolAddress failed at ufnvc_create");

    // the layout ufnvc_encode_chunk_dev gives its cudaMalloc'd scratch, sized for THIS call's n_chunks
    const ufnvc_config &c = h->cfg;
    const size_t G = size_t(c.lanes_per_substream / 32);
    const size_t n_sym = size_t(c.rows_per_substream) * h->w * c.c_y;
    const size_t steps = (n_sym + c.lanes_per_substream - 1) / c.lanes_per_substream;
    const size_t tmp_stride = steps * 32;
    const size_t stage_stride = (size_t(8) * G + G * 132 + 2 * steps * c.lanes_per_substream + 31) / 16 * 16;
    const size_t subs = size_t(n_chunks) * h->n_sub;
    const size_t tmp_bytes = align256(subs * G * tmp_stride * 2), stage_bytes = align256(subs * stage_stride), size_bytes = align256(subs * 4);
    const size_t need = tmp_bytes + stage_bytes + size_bytes;
    if (need > kStaticScratchBytes)
        return fail(h, UFNVC_E_INVALID_ARG, "ufnvc_encode_chunk_dev_static: this call needs " + std::to_string(need) +
                                                " bytes of scratch, the static array holds " + std::to_string(kStaticScratchBytes) +
                                                " (UFNVC_STATIC_SCRATCH_BYTES); use ufnvc_encode_chunk_dev or fewer chunks per call");

    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    unsigned char *base = static_cast<unsigned char *>(h->static_scratch);
    RansEncParams p{};
    p.idx = idx_dev; p.sym = sym_dev; p.cf = h->d_cf;
    p.n_chunks = n_chunks; p.n_sub = h->n_sub; p.h = h->h; p.w = h->w; p.c_y = c.c_y;
    p.rows_per_sub = c.rows_per_substream; p.W = c.lanes_per_substream; p.n_buckets = c.n_buckets;
    p.tmp_words = reinterpret_cast<uint16_t *>(base); p.tmp_stride = tmp_stride;
    p.stage = base + tmp_bytes; p.stage_stride = stage_stride;
    p.sizes = reinterpret_cast<uint32_t *>(base + tmp_bytes + stage_bytes);
    p.bits_out = bits_dev; p.cap = cap; p.sub_off = sub_off_dev; p.status = h->d_status;
    // the status word and the size table start at zero; everything else in the scratch is written before it is read
    cudaError_t e = cudaMemsetAsync(h->d_status, 0, 4, stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(p.sizes, 0, subs * 4, stream);
    if (e == cudaSuccess) e = launch_rans_encode(p, LaunchStream{stream, h->pdl});
    if (e != cudaSuccess) return fail(h, UFNVC_E_CUDA, std::string("ufnvc_encode_chunk_dev_static: ") + cudaGetErrorString(e));
    h->last_launches = 2;
    return UFNVC_OK;
}
