// C ABI of libufnvc (include/ufnvc.h): handle lifetime, validation, the launch sequence of the hot path.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>

#include "handle.h"

using namespace ufnvc;

namespace ufnvc {
int fail(ufnvc_handle *h, int code, const std::string &msg)
{
    if (h) h->err = msg;
    return code;
}
}  // namespace ufnvc

namespace {

const char *kNullHandleText = "null handle";

template <typename T> bool dev_alloc(ufnvc_handle *h, T *&p, size_t count)
{
    void *d = nullptr;
    if (cudaMalloc(&d, (count ? count : 1) * sizeof(T)) != cudaSuccess) return false;
    h->allocs.push_back(d);
    p = static_cast<T *>(d);
    return true;
}

int validate(const ufnvc_config &c, std::string &why)
{
#define BAD(cond, text) if (cond) { why = text; return UFNVC_E_BAD_CONFIG; }
    BAD(c.struct_size != sizeof(ufnvc_config), "struct_size mismatch");
    BAD(c.T < 1 || c.T > 64, "T out of range");
    BAD(c.height < 1 || c.width < 1 || c.height > 16384 || c.width > 16384, "frame size out of range");
    BAD(c.c_y < 8 || c.c_y % 8 || c.c_z < 16 || c.c_z % 16 || c.c_hyper < 16 || c.c_hyper % 16,
        "c_y must be a multiple of 8; c_z and c_hyper multiples of 16");
    BAD(c.c_trunk < 8 || c.c_trunk % 8, "c_trunk must be a multiple of 8");
    BAD(c.n_trunk_blocks < 0 || c.n_trunk_blocks > 64 || c.trunk_expand < 1, "bad trunk");
    BAD(c.dec_channels[0] != c.c_trunk || c.dec_channels[4] != 3, "dec_channels[0] must equal c_trunk and [4] must be 3");
    for (int s = 1; s < 4; ++s) BAD(c.dec_channels[s] < 8 || c.dec_channels[s] % 8, "dec_channels must be multiples of 8");
    BAD(c.n_buckets < 1 || c.n_buckets > 64, "n_buckets must be in [1,64]");
    BAD(!(c.scale_min > 0.0) || !(c.scale_max > c.scale_min), "need 0 < scale_min < scale_max");
    BAD(c.rows_per_substream < 1, "rows_per_substream >= 1");
    BAD(c.lanes_per_substream < 32 || c.lanes_per_substream % 32 || c.lanes_per_substream > 512, "lanes_per_substream: multiple of 32 in [32,512]");
    BAD(c.max_chunks_per_call < 1 || c.max_chunks_per_call > 64, "max_chunks_per_call out of range");
    BAD(c.weight_dtype != 0 && c.weight_dtype != 1, "weight_dtype must be 0 or 1");
    BAD(c.mu_steps != 1 && c.mu_steps != 4, "mu_steps must be 1 or 4");
    BAD(c.mu_steps == 4 && c.c_y % 32, "mu_steps == 4 needs c_y % 32 == 0 (the mean convs run on tensor cores only)");
    BAD(c.debug_flags & ~0x3FFu, "unknown debug_flags bit");
    BAD(c.n_ctx_blocks < 0 || c.n_ctx_blocks > 64, "n_ctx_blocks out of range");
    BAD(c.n_ctx_blocks > 0 && (c.c_trunk != 256 || (c.c_trunk * c.trunk_expand) % 128 || c.c_y % 64 || c.weight_dtype != 1 ||
                               c.c_hyper % 16 || c.c_z % 16),
        "a temporal context needs c_trunk == 256, c_y % 64 == 0, bf16 weights (the context generation runs on the fused tensor-core kernels)");
    BAD(c.n_ctx_blocks > 0 && (c.debug_flags & (UFNVC_DBG_FORCE_GENERIC | UFNVC_DBG_UNFUSED_TRUNK | UFNVC_DBG_PLAIN_DEPTHWISE)),
        "the context generation has no CUDA-core / unfused / plain-depthwise variant");
    BAD(c.n_enc_blocks < 0 || c.n_enc_blocks > 64, "n_enc_blocks out of range");
    BAD(c.n_enc_blocks > 0 && (c.c_trunk != 256 || (c.c_trunk * c.trunk_expand) % 128 || c.c_y % 32 || c.weight_dtype != 1 || c.mu_steps != 1 ||
                               c.c_y > 400),
        "the encoder needs c_trunk == 256, c_y % 32 == 0 (<= 400), bf16 weights and mu_steps == 1");
    BAD(c.n_enc_blocks > 0 && (c.debug_flags & (UFNVC_DBG_FORCE_GENERIC | UFNVC_DBG_UNFUSED_TRUNK | UFNVC_DBG_PLAIN_DEPTHWISE)),
        "the encoder has no CUDA-core / unfused / plain-depthwise variant");
    BAD(c.mu_steps == 4 && (c.debug_flags & UFNVC_DBG_FORCE_GENERIC), "mu_steps == 4 has no CUDA-core variant");
    // every kernel indexes latent elements and activation pixels with 32-bit integers (byte offsets are 64-bit)
    {
        const long long Hp = (c.height + 31) / 32 * 32, Wp = (c.width + 31) / 32 * 32, P = (Hp / 16) * (Wp / 16);
        const long long n = c.max_chunks_per_call;
        long long cmax = c.c_trunk * (long long)c.trunk_expand;
        BAD(n * P * c.c_y >= (1ll << 31), "max_chunks_per_call * h * w * c_y must stay below 2^31");
        BAD(n * c.T * P * cmax >= (1ll << 31), "max_chunks_per_call * T * h * w * c_trunk * trunk_expand must stay below 2^31");
        for (int s = 1; s <= 3; ++s) BAD(n * c.T * (P << (2 * s)) * c.dec_channels[s] >= (1ll << 31), "a decoder stage tensor must stay below 2^31 elements");
        BAD(n * c.T * 3 * (long long)c.height * c.width >= (1ll << 31), "the frame tensor must stay below 2^31 elements");
    }
#undef BAD
    return UFNVC_OK;
}

}  // namespace

extern "C" int ufnvc_create(const ufnvc_config *cfg, ufnvc_handle **out)
{
    if (!cfg || !out) return UFNVC_E_INVALID_ARG;
    std::string why;
    if (int rc = validate(*cfg, why)) return rc;
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return UFNVC_E_CUDA;
    if (prop.major != 10) return UFNVC_E_UNSUPPORTED_DEVICE;
    ufnvc_handle *h = new (std::nothrow) ufnvc_handle();
    if (!h) return UFNVC_E_OOM;
    h->cfg = *cfg;
    h->num_sms = prop.multiProcessorCount;
    h->H = (cfg->height + 31) / 32 * 32;
    h->W = (cfg->width + 31) / 32 * 32;
    h->h = h->H / 16;
    h->w = h->W / 16;
    h->h_z = (h->h + 3) / 4;
    h->w_z = (h->w + 3) / 4;
    h->n_sub = (h->h + cfg->rows_per_substream - 1) / cfg->rows_per_substream;
    h->n_sub_z = (h->h_z + cfg->rows_per_substream - 1) / cfg->rows_per_substream;
    h->max_chunks = cfg->max_chunks_per_call;
    h->has_ctx = cfg->n_ctx_blocks > 0;
    h->has_enc = cfg->n_enc_blocks > 0;
    h->c_cat = cfg->c_y + (h->has_ctx ? cfg->c_trunk : 0);
    const uint32_t dbg = cfg->debug_flags;
    h->force_generic = dbg & UFNVC_DBG_FORCE_GENERIC;
    h->use_fused_trunk = !(dbg & UFNVC_DBG_UNFUSED_TRUNK);
    h->use_pair_conv = h->use_pair_trunk = !(dbg & UFNVC_DBG_NO_CTA_PAIRS);
    h->pdl = !(dbg & UFNVC_DBG_NO_PDL);
    h->tail_fill = !(dbg & UFNVC_DBG_NO_TAIL_FILL);
    h->use_final_is = !(dbg & UFNVC_DBG_GENERIC_FINAL);
    h->use_dw_tma = !(dbg & UFNVC_DBG_PLAIN_DEPTHWISE);
    h->use_transposed_tiles = !(dbg & UFNVC_DBG_NO_TRANSPOSED_TILES);
    h->use_quad_clusters = !(dbg & UFNVC_DBG_NO_QUAD_CLUSTERS);
    h->hybrid_head = !(dbg & UFNVC_DBG_FP64_HEAD) && cfg->weight_dtype == 1 && cfg->c_y % 32 == 0 && cfg->c_hyper % 32 == 0 &&
                     !h->force_generic;
    // Error model of the tensor-core head (R12): ln sigma = sum of K = 9 * 2 c_hyper exact bf16 x bf16 products
    // accumulated in fp32.  (i) the 2-term split drops |x - hi - mid| <= 2^-16 |x| (two round-to-nearest steps to 8
    // significant bits, unit roundoff 2^-8 each); (ii) K fp32 additions: probabilistic rounding bound lambda sqrt(K) 2^-24 sum|terms| with lambda = 3.
    // sum |w||x| <= |w|_2 |x|_2 (Cauchy-Schwarz), so |error| <= kappa |w row|_2 |x patch|_2.
    h->head_kappa = std::ldexp(1.0, -16) + 3.0 * std::sqrt(18.0 * cfg->c_hyper) * std::ldexp(1.0, -24);
    // function attributes are per device: configure every kernel for the device this handle lives on
    if (configure_rans_kernels() != cudaSuccess || configure_hyper_kernels() != cudaSuccess || configure_depthwise_kernels() != cudaSuccess || configure_conv_tc_kernels() != cudaSuccess ||
        configure_trunk_kernels() != cudaSuccess || configure_final_kernels() != cudaSuccess) {
        cudaGetLastError();
        delete h;
        return UFNVC_E_CUDA;
    }
    // the no-allocation encoder's scratch lives in a __device__ array: its address on THIS device (a failure only disables
    // ufnvc_encode_chunk_dev_static, which then reports it)
    if (static_scratch_address(&h->static_scratch) != cudaSuccess) { cudaGetLastError(); h->static_scratch = nullptr; }

    // O3 tables + search accelerator
    build_cdf_tables(cfg->n_buckets, cfg->scale_min, cfg->scale_max, h->cdf32);
    std::vector<uint32_t> lut;
    std::vector<uint32_t> cf(h->cdf32.size(), 0u);
    build_search_lut(h->cdf32, cfg->n_buckets, lut);
    for (size_t i = 0; i < cf.size(); ++i)                                          // pos 255 is never a symbol
        if ((i & 255) != 255) cf[i] = h->cdf32[i] | ((h->cdf32[i + 1] - h->cdf32[i]) << 16);

    const size_t n = size_t(h->max_chunks), P = size_t(h->h) * h->w, Pz = size_t(h->h_z) * h->w_z, T = size_t(cfg->T);
    bool ok = dev_alloc(h, h->d_cf, cf.size()) && dev_alloc(h, h->d_lut, lut.size()) &&
              dev_alloc(h, h->hx1, n * Pz * cfg->c_hyper) &&
              dev_alloc(h, h->hx2, n * Pz * cfg->c_hyper) && dev_alloc(h, h->xs, n * Pz * 2 * cfg->c_hyper) && dev_alloc(h, h->xnorm2, n * Pz * size_t((cfg->c_hyper + 31) / 32)) &&
              dev_alloc(h, h->fix_list, n * P * cfg->c_y) && dev_alloc(h, h->mu, n * P * cfg->c_y) &&
              dev_alloc(h, h->lnscale, n * P * cfg->c_y) && dev_alloc(h, h->idx, n * P * cfg->c_y) &&
              dev_alloc(h, h->yhat, n * P * size_t(h->c_cat)) && dev_alloc(h, h->fa, n * T * P * cfg->c_trunk) &&
              dev_alloc(h, h->fb, n * T * P * cfg->c_trunk) &&
              dev_alloc(h, h->zero_block, 4 + size_t(cfg->n_trunk_blocks + std::max(cfg->n_ctx_blocks, cfg->n_enc_blocks) + 1) * ((n * T * P + 127) / 128 + 4)) &&
              dev_alloc(h, h->hidden, cfg->n_trunk_blocks ? n * T * P * cfg->c_trunk * cfg->trunk_expand : 1);
    if (ok) {      // everything a call clears up front sits in one block so that ONE memset node does it (decode.cu run())
        h->zero_words = 4 + size_t(cfg->n_trunk_blocks + std::max(cfg->n_ctx_blocks, cfg->n_enc_blocks) + 1) * ((n * T * P + 127) / 128 + 4);
        h->d_status = h->zero_block; h->fix_count = h->zero_block + 1; h->trunk_sync = h->zero_block + 4;
        ok = cudaMemset(h->zero_block, 0, h->zero_words * 4) == cudaSuccess;
    }
    if (ok && cfg->mu_steps == 4) {
        const size_t cs = (3 * size_t(cfg->c_y) + 63) / 64 * 64;       // [r | mu used | mu0 | zero pad], see weights.cu mu_net
        ok = dev_alloc(h, h->ymu[0], n * P * cs) && dev_alloc(h, h->ymu[1], n * P * cs) && dev_alloc(h, h->sym, n * P * cfg->c_y) &&
             cudaMemset(h->ymu[0], 0, n * P * cs * 2) == cudaSuccess && cudaMemset(h->ymu[1], 0, n * P * cs * 2) == cudaSuccess;
    }
    ok = ok && dev_alloc(h, h->z_idx, n * Pz * cfg->c_z) && dev_alloc(h, h->z_zero_mu, n * Pz * cfg->c_z) &&
         dev_alloc(h, h->z_scratch, n * Pz * cfg->c_z) && dev_alloc(h, h->z_hwc, n * Pz * cfg->c_z) &&
         dev_alloc(h, h->z_planar, n * Pz * cfg->c_z) && cudaMemset(h->z_zero_mu, 0, n * Pz * cfg->c_z * 4) == cudaSuccess;
    if (ok && (h->has_ctx || h->has_enc)) ok = dev_alloc(h, h->ca, n * P * cfg->c_trunk) && dev_alloc(h, h->cb, n * P * cfg->c_trunk);
    if (ok && h->has_ctx)
        ok = dev_alloc(h, h->ctx_q, n * Pz * cfg->c_hyper) &&
             cudaMemset(h->yhat, 0, n * P * size_t(h->c_cat) * 2) == cudaSuccess && cudaMemset(h->ctx_q, 0, n * Pz * cfg->c_hyper * 8) == cudaSuccess;
    if (ok && h->has_enc)
        ok = dev_alloc(h, h->p8, n * T * (P * 4) * 192) && dev_alloc(h, h->s2, n * T * P * 4 * cfg->c_trunk) && dev_alloc(h, h->ey, n * P * cfg->c_y) &&
             dev_alloc(h, h->henc_a, n * Pz * cfg->c_hyper) && dev_alloc(h, h->esym, n * P * cfg->c_y) && dev_alloc(h, h->ez, n * Pz * cfg->c_z);
    for (int s = 0; ok && s < 3; ++s) ok = dev_alloc(h, h->stage[s], n * T * (P << (2 * (s + 1))) * cfg->dec_channels[s + 1]);
    if (ok) ok = cudaMemcpy(h->d_cf, cf.data(), cf.size() * 4, cudaMemcpyHostToDevice) == cudaSuccess &&
                 cudaMemcpy(h->d_lut, lut.data(), lut.size() * 4, cudaMemcpyHostToDevice) == cudaSuccess &&
                 cudaMemset(h->d_status, 0, 4) == cudaSuccess;
    if (!ok) {
        cudaGetLastError();
        ufnvc_destroy(h);
        return UFNVC_E_OOM;
    }
    *out = h;
    return UFNVC_OK;
}

extern "C" int ufnvc_destroy(ufnvc_handle *h)
{
    if (!h) return UFNVC_E_INVALID_ARG;
    cudaDeviceSynchronize();
    for (void *p : h->allocs) cudaFree(p);
    for (void *p : h->weight_allocs) cudaFree(p);
    if (h->ev_made) for (auto &e : h->ev) cudaEventDestroy(e);
    for (auto &e : h->ev_dw) cudaEventDestroy(e);
    delete h;
    return UFNVC_OK;
}

extern "C" const char *ufnvc_last_error(const ufnvc_handle *h) { return h ? h->err.c_str() : kNullHandleText; }

extern "C" int ufnvc_get_status(ufnvc_handle *h, uint32_t *device_status)
{
    if (!h || !device_status) return UFNVC_E_INVALID_ARG;
    if (cudaMemcpy(device_status, h->d_status, 4, cudaMemcpyDeviceToHost) != cudaSuccess) return fail(h, UFNVC_E_CUDA, "status read failed");
    return UFNVC_OK;
}

extern "C" int ufnvc_debug_counter(ufnvc_handle *h, int which, uint64_t *value_host)
{
    if (!h || !value_host || which != 0) return UFNVC_E_INVALID_ARG;
    uint32_t v = 0;
    if (h->hybrid_head) {
        if (cudaDeviceSynchronize() != cudaSuccess || cudaMemcpy(&v, h->fix_count, 4, cudaMemcpyDeviceToHost) != cudaSuccess)
            return fail(h, UFNVC_E_CUDA, "cudaMemcpy(fix_count) failed");
    }
    *value_host = v;
    return UFNVC_OK;
}

extern "C" int ufnvc_get_cdf(const ufnvc_handle *h, uint32_t *cdf_host)
{
    if (!h || !cdf_host) return UFNVC_E_INVALID_ARG;
    std::memcpy(cdf_host, h->cdf32.data(), h->cdf32.size() * 4);
    return UFNVC_OK;
}

extern "C" int ufnvc_symbols_from_uniform(const ufnvc_handle *h, const uint8_t *idx_host, const uint16_t *u16_host, size_t n,
                                          int16_t *sym_host)
{
    if (!h || !idx_host || !u16_host || !sym_host) return UFNVC_E_INVALID_ARG;
    for (size_t i = 0; i < n; ++i) {
        if (idx_host[i] >= h->cfg.n_buckets) return UFNVC_E_INVALID_ARG;
        const uint32_t *c = &h->cdf32[size_t(idx_host[i]) * 256];
        int lo = 0, hi = 254;                      // largest p with c[p] <= u
        while (lo < hi) {
            const int mid = (lo + hi + 1) / 2;
            if (c[mid] <= u16_host[i]) lo = mid; else hi = mid - 1;
        }
        sym_host[i] = int16_t(lo - 127);
    }
    return UFNVC_OK;
}

extern "C" int ufnvc_convert_colour(const float *in_dev, float *out_dev, int n_img, int height, int width, int to_yuv, void *cuda_stream)
{
    if (!in_dev || !out_dev || n_img < 1 || height < 1 || width < 1) return UFNVC_E_INVALID_ARG;
    return launch_colour(in_dev, out_dev, (long long)height * width, n_img, to_yuv != 0, static_cast<cudaStream_t>(cuda_stream)) == cudaSuccess
               ? UFNVC_OK : UFNVC_E_CUDA;
}

extern "C" int ufnvc_get_z_prior_index(const ufnvc_handle *h, uint8_t *idx_host)
{
    if (!h || !idx_host) return UFNVC_E_INVALID_ARG;
    if (!h->z_prior_loaded) return UFNVC_E_NO_WEIGHTS;
    std::memcpy(idx_host, h->z_idx_c.data(), h->z_idx_c.size());
    return UFNVC_OK;
}

extern "C" long ufnvc_encode_z(const ufnvc_handle *h, const int16_t *z_host, uint8_t *bits_host, size_t cap, uint32_t *sub_off_host)
{
    if (!h || !z_host || !bits_host || !sub_off_host) return UFNVC_E_INVALID_ARG;
    if (!h->z_prior_loaded) return UFNVC_E_NO_WEIGHTS;
    const int cz = h->cfg.c_z, pz = h->h_z * h->w_z;
    std::vector<uint8_t> idx(size_t(pz) * cz);
    std::vector<int16_t> sym(size_t(pz) * cz);
    for (int p = 0; p < pz; ++p)
        for (int c = 0; c < cz; ++c) {                    // planar [c_z][pz] -> stream order (row, col, channel)
            idx[size_t(p) * cz + c] = h->z_idx_c[c];
            sym[size_t(p) * cz + c] = z_host[size_t(c) * pz + p];
        }
    size_t pos = 0;
    sub_off_host[0] = 0;
    for (int s = 0; s < h->n_sub_z; ++s) {
        const int r0 = s * h->cfg.rows_per_substream;
        const int rows = std::min(h->cfg.rows_per_substream, h->h_z - r0);
        const size_t e0 = size_t(r0) * h->w_z * cz, cnt = size_t(rows) * h->w_z * cz;
        const long nb = encode_substream(h->cdf32.data(), idx.data() + e0, sym.data() + e0, cnt, h->cfg.lanes_per_substream,
                                         bits_host + pos, cap - pos);
        if (nb < 0) return nb;
        pos += size_t(nb);
        sub_off_host[s + 1] = uint32_t(pos);
    }
    return long(pos);
}

extern "C" long ufnvc_encode_chunk(const ufnvc_handle *h, const uint8_t *idx_host, const int16_t *sym_host, uint8_t *bits_host,
                                   size_t cap, uint32_t *sub_off_host)
{
    if (!h || !idx_host || !sym_host || !bits_host || !sub_off_host) return UFNVC_E_INVALID_ARG;
    for (size_t i = 0, e = size_t(h->h) * h->w * h->cfg.c_y; i < e; ++i)
        if (idx_host[i] >= h->cfg.n_buckets) return UFNVC_E_INVALID_ARG;       // the tables hold n_buckets rows
    size_t pos = 0;
    sub_off_host[0] = 0;
    for (int s = 0; s < h->n_sub; ++s) {
        const int r0 = s * h->cfg.rows_per_substream;
        const int rows = std::min(h->cfg.rows_per_substream, h->h - r0);
        const size_t e0 = size_t(r0) * h->w * h->cfg.c_y, cnt = size_t(rows) * h->w * h->cfg.c_y;
        const long nb = encode_substream(h->cdf32.data(), idx_host + e0, sym_host + e0, cnt, h->cfg.lanes_per_substream,
                                         bits_host + pos, cap - pos);
        if (nb < 0) return nb;
        pos += size_t(nb);
        sub_off_host[s + 1] = uint32_t(pos);
    }
    return long(pos);
}
