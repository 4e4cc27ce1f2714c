// The launch sequence of ufnvc_chunk_decode: A1+A2 -> A3+A4 -> A5 -> B x (A6, A7) -> A8 -> A9.
// One host call, zero host synchronisations, everything on the caller's stream.
#include <algorithm>
#include <cmath>
#include <cstring>

#include "handle.h"

using namespace ufnvc;

namespace {

#define CU_TRY(expr)                                                                                         \
    do {                                                                                                     \
        cudaError_t e__ = (expr);                                                                            \
        if (e__ != cudaSuccess) return fail(h, UFNVC_E_CUDA, std::string(#expr) + ": " + cudaGetErrorString(e__)); \
    } while (0)

// conv dispatch: tcgen05 implicit GEMM when the layer and the activation map qualify, CUDA-core kernel otherwise.
cudaError_t conv(ufnvc_handle *h, const ConvLayer &L, const ConvProblem &P, const ufnvc_handle::ActMap &am, const EpiParams &E,
                 LaunchStream st, int *launches)
{
    if (launches) ++*launches;
    if (L.use_tc && L.taps == 9 && am.halo_ok && !h->force_generic && h->use_pair_conv && L.has_half_map &&
        (E.mode == EPI_PS2 || E.mode == EPI_MU) && P.W > 8)
        return launch_conv_halo_pair(L, P, am.halo_t ? am.tm_halo_t : am.tm_halo, E, h->num_sms, st, am.halo_t);
    if (L.use_tc && L.taps == 9 && am.halo_ok && !h->force_generic)
        return launch_conv_halo(L, P, am.tm_halo, E, h->num_sms, st);
    if (L.use_tc && am.ok && !h->force_generic) return launch_conv_tc(L, P, am.tm, am.tile_h, am.tile_w, am.flat, E, h->num_sms, st);
    return launch_conv_generic(L, P, E, st);
}

struct Stage { cudaEvent_t *ev; int i; cudaEvent_t *dw; };   // dw: one event after every depthwise launch (A6 / A7 split)
inline void mark(Stage *s, cudaStream_t st) { if (s) cudaEventRecord(s->ev[s->i++], st); }

int run(ufnvc_handle *h, int n, const int16_t *z, const uint8_t *bits, size_t bits_bytes, const uint32_t *sub_off, float *frames,
        cudaStream_t stream, const uint8_t *idx_ovr, const float *mu_ovr, const ufnvc_taps *taps, bool entropy_params_only,
        float *mu_out, float *ls_out, uint8_t *idx_out, Stage *sg, int *launches)
{
    const ufnvc_config &c = h->cfg;
    const LaunchStream st{stream, h->pdl};
    int local_launches = 0;                    // kernels of this library enqueued by this call (memsets / copies not counted)
    if (!launches) launches = &local_launches;
    struct Publish { ufnvc_handle *h; int *n; ~Publish() { h->last_launches = *n; } } publish{h, launches};
    const int P = h->h * h->w, Pz = h->h_z * h->w_z;
    const size_t ne = size_t(n) * P * c.c_y;

    // everything the call clears (status word, the head's fix-up count, the trunk's tile counters) is cleared up front by ONE
    // memset, so that no memset node sits between kernels launched with programmatic stream serialization
    {
        // [status | fix_count | pad | trunk counters]: the status word is skipped when an earlier call's status is kept, the
        // trunk counters when this call does not reach the trunk
        const bool keep = entropy_params_only || h->keep_status;
        const bool trunk = !entropy_params_only && frames && c.n_trunk_blocks > 0 && h->tail_fill;
        const bool trunk_or_ctx = !entropy_params_only && frames && (c.n_trunk_blocks > 0 || h->has_ctx) && h->tail_fill;
        const size_t words = (trunk || trunk_or_ctx) ? 4 + size_t(c.n_trunk_blocks + c.n_ctx_blocks) * h->trunk_sync_stride : 4;
        CU_TRY(cudaMemsetAsync(h->zero_block + (keep ? 1 : 0), 0, (words - (keep ? 1 : 0)) * 4, st));
    }
    // ---- A1 + A2: hyper-decoder in fp64 -> mu, ln sigma, bucket index ----
    const bool need_hyper = entropy_params_only || !idx_ovr || !mu_ovr || (taps && (taps->mu || taps->lnscale));
    mark(sg, st);
    if (need_hyper) {
        // layer 0 reads the int16 hyper-latent directly; layers 0 and 1 are one fp64 launch each (hyper.cu)
        CU_TRY(launch_hyper_conv(h->hyper[0], z, true, h->hx1, n, h->h_z, h->w_z, st));
        HeadParams hp{c.c_y, h->h, h->w, c.n_buckets, std::log(c.scale_min), std::log(c.scale_max), h->mu, h->lnscale, h->idx};
        const double *q = h->has_ctx ? h->ctx_q : nullptr;
        if (h->hybrid_head && h->am_xs.ok && h->head_tc.use_tc) {
            // layer 1 also emits the bf16 hi|mid split; the head runs on tensor cores; elements whose ln sigma may land on the
            // wrong side of a bucket edge are re-decided in fp64 (identical decisions to the all-fp64 path, R12)
            CU_TRY(launch_hyper_conv(h->hyper[1], h->hx1, false, h->hx2, n, h->h_z, h->w_z, st, h->xs, h->xnorm2, q));
            const double step = (hp.ln_hi - hp.ln_lo) / double(c.n_buckets - 1 > 0 ? c.n_buckets - 1 : 1);
            EpiParams E{};
            E.mode = EPI_HEAD; E.act = ACT_NONE;
            E.mu = h->mu; E.lnscale = h->lnscale; E.idx = h->idx; E.fix_list = h->fix_list; E.fix_count = h->fix_count;
            E.c_y = c.c_y; E.lat_h = h->h; E.lat_w = h->w; E.n_buckets = c.n_buckets;
            E.ln_lo = float(hp.ln_lo); E.ln_hi = float(hp.ln_hi); E.t_scale = float(1.0 / step);
            E.wnorm = h->head_wnorm; E.xnorm2 = h->xnorm2; E.xnorm_parts = hyper_xnorm_parts(h->hyper[1]); E.kappa_t = float(h->head_kappa / step);
            ConvProblem pr{h->xs, n, h->h_z, h->w_z, 1};
            // The head is bound by L2 -> SM weight traffic (18.9 MB of weights, re-read once per M tile): the CTA-pair halo
            // kernel shares every weight tile between two 16 x 8 pixel tiles (M = 256) and loads the activations once per
            // slab instead of once per tap.  Fallback: the shifted-TMA-box kernel (narrow maps, debug flag).
            if (h->use_pair_conv && h->head_tc.has_half_map && h->am_xs.halo_ok && h->w_z > 8)
                CU_TRY(launch_conv_halo_pair(h->head_tc, pr, h->am_xs.halo_t ? h->am_xs.tm_halo_t : h->am_xs.tm_halo, E, h->num_sms, st, h->am_xs.halo_t));
            else
                CU_TRY(launch_conv_tc(h->head_tc, pr, h->am_xs.tm, h->am_xs.tile_h, h->am_xs.tile_w, false, E, h->num_sms, st));
            CU_TRY(launch_hyper_fix(h->fix_list, h->fix_count, h->hx2, h->head_fix_w, h->head_fix_b, c.c_hyper, h->h_z, h->w_z, hp,
                                    h->num_sms, st));
            *launches += 4;                    // two fp64 layers + head conv + fp64 fix
        } else {
            CU_TRY(launch_hyper_conv(h->hyper[1], h->hx1, false, h->hx2, n, h->h_z, h->w_z, st, nullptr, nullptr, q));
            CU_TRY(launch_hyper_head(h->hyper[2], h->hx2, n, h->h_z, h->w_z, hp, st));
            *launches += 3;
        }
    }
    if (entropy_params_only) {
        if (mu_out) CU_TRY(cudaMemcpyAsync(mu_out, h->mu, ne * 4, cudaMemcpyDeviceToDevice, st));
        if (ls_out) CU_TRY(cudaMemcpyAsync(ls_out, h->lnscale, ne * 4, cudaMemcpyDeviceToDevice, st));
        if (idx_out) CU_TRY(cudaMemcpyAsync(idx_out, h->idx, ne, cudaMemcpyDeviceToDevice, st));
        return UFNVC_OK;
    }
    const uint8_t *idx = idx_ovr ? idx_ovr : h->idx;
    const float *mu = mu_ovr ? mu_ovr : h->mu;
    if (taps) {
        if (taps->mu) CU_TRY(cudaMemcpyAsync(taps->mu, mu, ne * 4, cudaMemcpyDeviceToDevice, st));
        if (taps->lnscale) CU_TRY(cudaMemcpyAsync(taps->lnscale, h->lnscale, ne * 4, cudaMemcpyDeviceToDevice, st));
        if (taps->idx) CU_TRY(cudaMemcpyAsync(taps->idx, idx, ne, cudaMemcpyDeviceToDevice, st));
    }
    mark(sg, st);

    // ---- A3 + A4: rANS decode + dequantisation ----
    RansParams rp{};
    rp.bits = bits; rp.bits_bytes = bits_bytes; rp.sub_off = sub_off; rp.idx = idx; rp.mu = mu;
    rp.sub_stride = h->y_sub_stride > 0 ? h->y_sub_stride : h->n_sub; rp.sub_first = h->y_sub_stride > 0 ? h->n_sub_z : 0;
    rp.cf = h->d_cf; rp.lut = h->d_lut;
    rp.n_chunks = n; rp.n_sub = h->n_sub; rp.h = h->h; rp.w = h->w; rp.c_y = c.c_y;
    rp.rows_per_sub = c.rows_per_substream; rp.W = c.lanes_per_substream; rp.n_buckets = c.n_buckets;
    rp.y_stride = h->c_cat;
    const bool progressive = c.mu_steps == 4;
    rp.yhat = h->yhat; rp.sym_tap = progressive ? h->sym : (taps ? taps->sym : nullptr); rp.yhat_tap = taps ? taps->yhat : nullptr;
    rp.status = h->d_status;
    CU_TRY(launch_rans_decode(rp, st));
    *launches += 1;                            // rANS decode
    if (progressive) {
        // ---- NEXT-1 (R21): four-step progressive means, no bit-stream contact.  The rANS kernel has
        // written r (h->sym) and r + mu0 (taps); step 0 keeps that on partition 0, steps 1..3 are 3x3 convs over
        // [y decoded so far ; mu0] (y as the pair r, mu: mu_steps.cu) whose epilogue switches partition k on.  The last
        // step writes the dense y that A5 reads.
        if (taps && taps->sym) CU_TRY(cudaMemcpyAsync(taps->sym, h->sym, ne * 2, cudaMemcpyDeviceToDevice, st));
        const int cs = h->mu_net[0].c_in;       // [r | mu used | mu0 | pad] channels per pixel
        CU_TRY(launch_mu_prep(h->sym, mu, h->ymu[0], h->ymu[1], n, h->h, h->w, c.c_y, cs, st));
        *launches += 1;
        for (int k = 1; k <= 3; ++k) {
            const int src = (k - 1) & 1;
            ConvProblem pr{h->ymu[src], n, h->h, h->w, 1};
            EpiParams E{};
            E.mode = EPI_MU; E.act = ACT_NONE;
            E.out = k < 3 ? static_cast<void *>(h->ymu[k & 1]) : static_cast<void *>(h->yhat);
            E.out_stride = k < 3 ? cs : h->c_cat;
            E.y_in = h->ymu[src]; E.in_stride = cs;
            E.sym = h->sym; E.c_y = c.c_y; E.mu_step = k; E.mu_last = k == 3;
            E.mu_tap = taps ? taps->mu : nullptr; E.yhat_tap = taps ? taps->yhat : nullptr;
            CU_TRY(conv(h, h->mu_net[k - 1], pr, h->am_ymu[src], E, st, launches));
        }
    }
    mark(sg, st);
    if (!frames) return UFNVC_OK;

    // ---- A5: cross-frame unfold, 1x1 conv c_y -> T*c_trunk, channel t*c_trunk + c -> frame t ----
    const int T = c.T, Ct = c.c_trunk;
    const size_t fe = size_t(n) * T * P * Ct;
    {
        ConvProblem pr{h->yhat, n, h->h, h->w, 1};
        EpiParams E{EPI_NHWC, ACT_NONE, h->fa, nullptr, Ct, (long long)P * Ct, (long long)T * P * Ct, 0, 0, 0};
        CU_TRY(conv(h, h->xframe, pr, h->am_yhat, E, st, launches));
    }
    if (taps && taps->f0) CU_TRY(cudaMemcpyAsync(taps->f0, h->fa, fe * 2, cudaMemcpyDeviceToDevice, st));
    mark(sg, st);

    // ---- A6 + A7: trunk of residual DC blocks, weights shared over t (t is batch) ----
    const int Ce = Ct * c.trunk_expand;
    for (int k = 0; k < c.n_trunk_blocks; ++k) {
        const ufnvc_handle::TrunkBlock &tb = h->trunk[k];
        // every block must be fused for the counters to be produced where the next depthwise kernel expects them
        bool fused_ok = h->use_fused_trunk && !h->force_generic;
        for (const auto &t2 : h->trunk) fused_ok = fused_ok && t2.fused.ok;
        if (sg && sg->dw) { cudaEventRecord(sg->dw[2 * k + 1], st); }
        // tail filling: block k's depthwise tiles wait for the MLP tiles of block k - 1 that cover their halo
        // box instead of for the whole MLP grid, and are handed out by a per-block counter
        uint32_t *sync_k = h->trunk_sync + size_t(k) * h->trunk_sync_stride;
        const bool mlp_counts = fused_ok && trunk_counts_tiles((long long)n * T * P, h->use_pair_trunk) && h->tail_fill;
        if (h->dw_tma_ok) CU_TRY(launch_dwconv3x3_tma(h->tm_dw, h->fb, tb.dw_w, tb.dw_b, n * T, h->h, h->w, Ct, h->num_sms, st, h->tail_fill ? sync_k : nullptr,
                                                      (k > 0 && mlp_counts) ? sync_k - h->trunk_sync_stride + 1 : nullptr));
        else CU_TRY(launch_dwconv3x3(h->fa, h->fb, tb.dw_w, tb.dw_b, n * T, h->h, h->w, Ct, st));
        if (launches) ++*launches;
        if (sg && sg->dw) { cudaEventRecord(sg->dw[2 * k], st); }
        if (fused_ok) {
            CU_TRY(launch_trunk_mlp(tb.fused, tb.pw1, tb.pw2, h->fa, h->fa, (long long)n * T * P, h->num_sms, h->use_pair_trunk, st,
                                    mlp_counts ? sync_k + 1 : nullptr, h->use_quad_clusters));
            if (launches) ++*launches;
            continue;
        }
        ConvProblem p1{h->fb, n * T, h->h, h->w, 1};
        EpiParams E1{EPI_NHWC, ACT_GELU, h->hidden, nullptr, Ce, 0, (long long)P * Ce, 0, 0, 0};
        CU_TRY(conv(h, tb.pw1, p1, h->am_fb, E1, st, launches));
        ConvProblem p2{h->hidden, n * T, h->h, h->w, 1};
        EpiParams E2{EPI_NHWC, ACT_NONE, h->fa, h->fa, Ct, 0, (long long)P * Ct, 0, 0, 0};
        CU_TRY(conv(h, tb.pw2, p2, h->am_hidden, E2, st, launches));
    }
    if (taps && taps->trunk) CU_TRY(cudaMemcpyAsync(taps->trunk, h->fa, fe * 2, cudaMemcpyDeviceToDevice, st));
    mark(sg, st);    // (A6 and A7 are reported together here; the profiled call splits them with its own events)

    // ---- A8: frame-specific decoders, stages 1..3, one grouped launch over t per stage ----
    const bf16 *x = h->fa;
    const ufnvc_handle::ActMap *am = &h->am_fa;
    int sh = h->h, sw = h->w;
    for (int s = 0; s < 3; ++s) {
        const int co = c.dec_channels[s + 1];
        ConvProblem pr{x, n * T, sh, sw, T};
        pr.reverse = (s & 1) == 0;         // trunk forwards, stage 1 backwards, 2 forwards, 3 backwards, A9 forwards: each kernel
                                           // starts on the data its predecessor wrote last, which is still in L2
        EpiParams E{EPI_PS2, ACT_GELU, h->stage[s], nullptr, 0, 0, (long long)sh * sw * 4 * co, co, 0, 0};
        CU_TRY(conv(h, h->dec[s], pr, *am, E, st, launches));
        sh *= 2; sw *= 2;
        x = h->stage[s];
        am = &h->am_stage[s];
        if (taps && taps->stage[s]) CU_TRY(cudaMemcpyAsync(taps->stage[s], x, size_t(n) * T * sh * sw * co * 2, cudaMemcpyDeviceToDevice, st));
    }
    mark(sg, st);

    // ---- A9: last stage (linear) + pixel-shuffle + clamp + crop + planar fp32 ----
    {
        if (h->final_is.ok && !h->force_generic) {
            CU_TRY(launch_final_is(h->final_is, h->dec[3], n * T, sh, sw, frames, c.height, c.width, h->num_sms, st));
            ++*launches;
        } else {
            ConvProblem pr{x, n * T, sh, sw, T};
            EpiParams E{EPI_FINAL, ACT_NONE, frames, nullptr, 0, 0, (long long)3 * c.height * c.width, 3, c.height, c.width};
            CU_TRY(conv(h, h->dec[3], pr, *am, E, st, launches));
        }
    }
    mark(sg, st);

    // ---- NEXT-2a (R23): context generation, C_{i+1} = bf16(conv_out(DCblock^{B_c}(conv_fold([F_i[0]; ..; F_i[T-1]])))), then its
    // prior branch q.  F_i is the trunk's output, still in fa.  The new state overwrites the context block of the [y ; C]
    // buffer, which nothing of this call reads any more (A5 consumed it; every kernel of the chain waits for its predecessor).
    if (h->has_ctx) {
        {
            ConvProblem pr{h->fa, n, h->h, h->w, 1, true};
            EpiParams E{EPI_NHWC, ACT_NONE, h->ca, nullptr, Ct, 0, (long long)P * Ct, 0, 0, 0};
            CU_TRY(conv(h, h->ctx_fold, pr, h->am_fa, E, st, launches));
        }
        for (int k = 0; k < c.n_ctx_blocks; ++k) {
            const ufnvc_handle::TrunkBlock &tb = h->ctx_blocks[k];
            uint32_t *sync_k = h->trunk_sync + size_t(c.n_trunk_blocks + k) * h->trunk_sync_stride;
            const bool mlp_counts = trunk_counts_tiles((long long)n * P, h->use_pair_trunk) && h->tail_fill;
            CU_TRY(launch_dwconv3x3_tma(h->tm_dw_ctx, h->cb, tb.dw_w, tb.dw_b, n, h->h, h->w, Ct, h->num_sms, st, h->tail_fill ? sync_k : nullptr,
                                        (k > 0 && mlp_counts) ? sync_k - h->trunk_sync_stride + 1 : nullptr));
            CU_TRY(launch_trunk_mlp(tb.fused, tb.pw1, tb.pw2, h->ca, h->ca, (long long)n * P, h->num_sms, h->use_pair_trunk, st,
                                    mlp_counts ? sync_k + 1 : nullptr, h->use_quad_clusters));
            *launches += 2;
        }
        {
            ConvProblem pr{h->ca, n, h->h, h->w, 1};
            EpiParams E{EPI_NHWC, ACT_NONE, h->yhat + c.c_y, nullptr, Ct, 0, (long long)P * h->c_cat, 0, 0, 0};
            E.pix_stride = h->c_cat;
            CU_TRY(conv(h, h->ctx_out, pr, h->am_ca, E, st, launches));
        }
        CU_TRY(launch_ctx_prior(h->yhat + c.c_y, h->c_cat, Ct, h->ctx_prior_w, h->ctx_prior_b, h->ctx_q, n, h->h, h->w, h->h_z, h->w_z, c.c_hyper, st));
        ++*launches;
    }
    mark(sg, st);
    return UFNVC_OK;
}

int check_call(ufnvc_handle *h, int n_chunks, const void *z, const void *bits, const void *sub_off)
{
    if (!h) return UFNVC_E_INVALID_ARG;
    if (!h->weights_loaded) return fail(h, UFNVC_E_NO_WEIGHTS, "ufnvc_load_weights has not succeeded on this handle");
    if (n_chunks < 1 || n_chunks > h->max_chunks) return fail(h, UFNVC_E_INVALID_ARG, "n_chunks outside [1, max_chunks_per_call]");
    if (!z || !bits || !sub_off) return fail(h, UFNVC_E_INVALID_ARG, "null device pointer");
    if (reinterpret_cast<uintptr_t>(bits) & 3) return fail(h, UFNVC_E_INVALID_ARG, "bits_dev must be 4-byte aligned");
    return UFNVC_OK;
}

}  // namespace

// choose the 128-pixel tile (TH x TW) that covers an H x W image with the fewest tiles; ties -> wider rows
static void pick_tile(int H, int W, int &th, int &tw)
{
    long best = -1;
    for (int t = 1; t <= 16; t *= 2) {
        const int w = 128 / t;
        const long tiles = long((H + t - 1) / t) * ((W + w - 1) / w);
        if (best < 0 || tiles < best) { best = tiles; th = t; tw = w; }
    }
}

static bool make_act_map(ufnvc_handle *h, ufnvc_handle::ActMap &am, const bf16 *base, int n_img, int H, int W, int C, bool want_flat,
                         int imgs_per_chunk)
{
    am.ok = false;
    am.halo_ok = false;
    if (C % 64) return true;
    std::string err;
    am.flat = want_flat && ((long long)imgs_per_chunk * H * W) % 128 == 0;
    if (am.flat) {
        am.tile_h = 1; am.tile_w = 128;
        if (!tc_make_act_tmap(&am.tm, base, 1, int((long long)n_img * H * W / 128), 128, C, 1, 128, err)) { h->err = err; return false; }
    } else {
        pick_tile(H, W, am.tile_h, am.tile_w);
        if (!tc_make_act_tmap(&am.tm, base, n_img, H, W, C, am.tile_h, am.tile_w, err)) { h->err = err; return false; }
        if (!tc_make_halo_tmap(&am.tm_halo, base, n_img, H, W, C, err)) { h->err = err; return false; }
        am.halo_ok = true;
        am.halo_t = false;
        if (halo_prefers_transposed(H, W) && h->use_transposed_tiles) {
            if (!tc_make_halo_tmap_transposed(&am.tm_halo_t, base, n_img, H, W, C, err)) { h->err = err; return false; }
            am.halo_t = true;
        }
    }
    am.ok = true;
    return true;
}

extern "C" int ufnvc_load_weights(ufnvc_handle *h, const void *blob_host, size_t bytes)
{
    if (!h || !blob_host) return UFNVC_E_INVALID_ARG;
    h->weights_loaded = false;
    if (int rc = load_weights_impl(h, blob_host, bytes)) return rc;
    // tcgen05 path: weight descriptors + descriptors of the (fixed) workspace activations
    const ufnvc_config &c = h->cfg;
    std::string err;
    bool ok = tc_make_weight_tmap(h->xframe, err, 0);
    if (h->hybrid_head) {
        // N tile of the hyper head conv: the z map is tiny (510 pixels at 1080p = 4-6 M tiles), so with the widest N tile
        // (256) fewer tiles than SMs exist and each CTA runs one long tile with its epilogue exposed; 128 doubles the tile
        // count (measured at 1080p: A1+A2 98 -> 93 us; 64 and 32 are slower again).
        const long long m_tiles = ((long long)h->max_chunks * h->h_z * h->w_z + 127) / 128;
        const int auto_bn = (h->head_tc.n_pad % 128 == 0 && m_tiles * (h->head_tc.n_pad / 256) < h->num_sms) ? 128 : 0;
        ok = ok && tc_make_weight_tmap(h->head_tc, err, auto_bn);
    }
    for (auto &tb : h->trunk) ok = ok && tc_make_weight_tmap(tb.pw1, err) && tc_make_weight_tmap(tb.pw2, err);
    for (int s = 0; s < 4; ++s) ok = ok && tc_make_weight_tmap(h->dec[s], err);
    if (h->has_ctx) {
        // the fold over T has K = T c_trunk on only h w / 128 pixel tiles per chunk: halve the n tile when that leaves SMs without
        // work (each CTA then streams half the weight bytes of its long K loop)
        const int fold_bn = (long long)h->max_chunks * h->h * h->w / 128 * (c.c_trunk / 256) <= h->num_sms / 2 ? 128 : 0;
        ok = ok && tc_make_weight_tmap(h->ctx_fold, err, fold_bn) && tc_make_weight_tmap(h->ctx_out, err);
        for (auto &tb : h->ctx_blocks) ok = ok && tc_make_weight_tmap(tb.pw1, err) && tc_make_weight_tmap(tb.pw2, err);
    }
    // progressive means: three small 3x3 convs in a row on the latent map -- n tiles of 64 on the CTA-pair kernel when that puts a
    // unit on (nearly) every pair instead of one 128-wide tile on half of the SMs
    for (int k = 0; k < 3 && c.mu_steps == 4; ++k) {
        const long pairs = ((long(h->h + 15) / 16) * ((h->w + 7) / 8) + 1) / 2 * h->max_chunks;
        const int mu_bn = (h->mu_net[k].n_pad % 64 == 0 && pairs * (h->mu_net[k].n_pad / 64) <= h->num_sms / 2 + 8) ? 64 : 0;
        ok = ok && tc_make_weight_tmap(h->mu_net[k], err, mu_bn);
    }
    if (!ok) return fail(h, UFNVC_E_CUDA, err);
    const int n = h->max_chunks, T = c.T;
    if (h->hybrid_head) ok = make_act_map(h, h->am_xs, h->xs, n, h->h_z, h->w_z, 2 * c.c_hyper, false, 1);
    ok = ok && make_act_map(h, h->am_yhat, h->yhat, n, h->h, h->w, h->c_cat, true, 1) &&
         make_act_map(h, h->am_fb, h->fb, n * T, h->h, h->w, c.c_trunk, true, T) &&
         make_act_map(h, h->am_hidden, h->hidden, n * T, h->h, h->w, c.c_trunk * c.trunk_expand, true, T) &&
         make_act_map(h, h->am_fa, h->fa, n * T, h->h, h->w, c.c_trunk, false, T);
    if (c.mu_steps == 4) {
        for (int b = 0; ok && b < 2; ++b) ok = make_act_map(h, h->am_ymu[b], h->ymu[b], n, h->h, h->w, h->mu_net[0].c_in, false, 1);
        if (ok && (!h->am_ymu[0].ok || !h->mu_net[0].use_tc || h->force_generic))
            return fail(h, UFNVC_E_BAD_CONFIG, "mu_steps == 4 needs the tensor-core conv path (c_y % 32 == 0, no UFNVC_DBG_FORCE_GENERIC)");
    }
    h->trunk_sync_stride = size_t(((long long)n * T * h->h * h->w + 127) / 128 + 4);
    h->dw_tma_ok = false;
    if (ok && c.n_trunk_blocks > 0 && c.c_trunk % 64 == 0 && c.c_trunk <= 256 && h->use_dw_tma) {
        ok = tc_make_act_tmap(&h->tm_dw, h->fa, n * T, h->h, h->w, c.c_trunk, 10, 10, h->err, /*swizzle=*/false);
        h->dw_tma_ok = ok;
    }
    for (auto &tb : h->trunk)
        if (ok && !trunk_make_maps(tb.fused, h->fb, (long long)n * T * h->h * h->w, tb.pw1, tb.pw2, h->err)) ok = false;
    if (ok && (h->has_ctx || h->has_enc))
        ok = make_act_map(h, h->am_ca, h->ca, n, h->h, h->w, c.c_trunk, false, 1) &&
             tc_make_act_tmap(&h->tm_dw_ctx, h->ca, n, h->h, h->w, c.c_trunk, 10, 10, h->err, /*swizzle=*/false);
    if (ok && h->has_enc) {
        // encoder (R24): patches [n T][H/8][W/8][192], embedded + space-to-depth x2 [n T][h][w][4 c_trunk]
        const int fold_bn = (long long)h->max_chunks * h->h * h->w / 128 * (c.c_trunk / 256) <= h->num_sms / 2 ? 128 : 0;
        ok = tc_make_weight_tmap(h->enc_patch, err) && tc_make_weight_tmap(h->enc_fold, err, fold_bn) && tc_make_weight_tmap(h->enc_y, err);
        for (auto &tb : h->enc_blocks) ok = ok && tc_make_weight_tmap(tb.pw1, err) && tc_make_weight_tmap(tb.pw2, err);
        if (!ok) return fail(h, UFNVC_E_CUDA, err);
        ok = make_act_map(h, h->am_p8, h->p8, n * T, 2 * h->h, 2 * h->w, 192, false, T) &&
             make_act_map(h, h->am_s2, h->s2, n * T, h->h, h->w, 4 * c.c_trunk, false, T);
        for (auto &tb : h->enc_blocks)
            if (ok && (!trunk_make_maps(tb.fused, h->cb, (long long)n * h->h * h->w, tb.pw1, tb.pw2, h->err) || !tb.fused.ok)) ok = false;
        if (ok && h->has_ctx) {
            // E3 reads the context block of the [y ; C] buffer in place: a tensor map with the buffer's pixel stride
            ok = tc_make_weight_tmap(h->enc_ctx, err);
            if (!ok) return fail(h, UFNVC_E_CUDA, err);
            pick_tile(h->h, h->w, h->am_cin.tile_h, h->am_cin.tile_w);
            h->am_cin.flat = false;
            ok = tc_make_act_tmap(&h->am_cin.tm, h->yhat + c.c_y, n, h->h, h->w, c.c_trunk, h->am_cin.tile_h, h->am_cin.tile_w, h->err, true, h->c_cat);
            h->am_cin.ok = ok;
        }
        if (ok && (!h->am_p8.ok || !h->am_s2.ok || !h->am_ca.ok || !h->enc_patch.use_tc || !h->enc_fold.use_tc || !h->enc_y.use_tc)) {
            ok = false; h->err = "the encoder needs the tensor-core conv path";
        }
    }
    if (ok && h->has_ctx) {
        for (auto &tb : h->ctx_blocks)
            if (ok && (!trunk_make_maps(tb.fused, h->cb, (long long)n * h->h * h->w, tb.pw1, tb.pw2, h->err) || !tb.fused.ok)) ok = false;
        if (ok && (!h->am_fa.ok || !h->ctx_fold.use_tc || !h->ctx_out.use_tc || !h->am_ca.ok)) { ok = false; h->err = "context generation needs the tensor-core conv path"; }
    }
    for (int s = 0; ok && s < 3; ++s)
        ok = make_act_map(h, h->am_stage[s], h->stage[s], n * T, h->h << (s + 1), h->w << (s + 1), c.dec_channels[s + 1], false, T);
    h->final_is.ok = false;
    if (ok && h->use_final_is && c.dec_channels[3] % 64 == 0)
        ok = final_make_maps(h->final_is, h->dec[3], h->stage[2], n * T, h->h << 3, h->w << 3, c.width, h->err);
    if (!ok) return fail(h, UFNVC_E_CUDA, h->err);
    h->weights_loaded = true;
    return UFNVC_OK;
}

extern "C" int ufnvc_chunk_decode_ex(ufnvc_handle *h, int n_chunks, const int16_t *z_dev, const uint8_t *bits_dev, size_t bits_bytes,
                                     const uint32_t *sub_off_dev, float *frames_dev, void *cuda_stream, const uint8_t *idx_override_dev,
                                     const float *mu_override_dev, const ufnvc_taps *taps)
{
    if (int rc = check_call(h, n_chunks, z_dev, bits_dev, sub_off_dev)) return rc;
    if (taps && taps->struct_size != sizeof(ufnvc_taps)) return fail(h, UFNVC_E_INVALID_ARG, "ufnvc_taps.struct_size mismatch");
    return run(h, n_chunks, z_dev, bits_dev, bits_bytes, sub_off_dev, frames_dev, static_cast<cudaStream_t>(cuda_stream),
               idx_override_dev, mu_override_dev, taps, false, nullptr, nullptr, nullptr, nullptr, nullptr);
}

extern "C" int ufnvc_chunk_decode(ufnvc_handle *h, int n_chunks, const int16_t *z_dev, const uint8_t *bits_dev, size_t bits_bytes,
                                  const uint32_t *sub_off_dev, float *frames_dev, void *cuda_stream)
{
    if (int rc = check_call(h, n_chunks, z_dev, bits_dev, sub_off_dev)) return rc;
    if (!frames_dev) return fail(h, UFNVC_E_INVALID_ARG, "frames_dev is null");
    return run(h, n_chunks, z_dev, bits_dev, bits_bytes, sub_off_dev, frames_dev, static_cast<cudaStream_t>(cuda_stream), nullptr,
               nullptr, nullptr, false, nullptr, nullptr, nullptr, nullptr, nullptr);
}

// ---- NEXT-3 (R22): the hyper-latent from bytes ------------------------------------------------------------------
namespace {
int decode_z_impl(ufnvc_handle *h, int n, const uint8_t *bits, size_t bits_bytes, const uint32_t *sub_off, int sub_stride,
                  int16_t *z_planar_out, cudaStream_t stream, int *launches)
{
    const ufnvc_config &c = h->cfg;
    const LaunchStream st{stream, h->pdl};
    if (!h->z_prior_loaded) return fail(h, UFNVC_E_NO_WEIGHTS, "the weights blob holds no zprior.lnscale tensor");
    CU_TRY(cudaMemsetAsync(h->d_status, 0, 4, st));
    RansParams rp{};
    rp.bits = bits; rp.bits_bytes = bits_bytes; rp.sub_off = sub_off; rp.sub_stride = sub_stride; rp.sub_first = 0;
    rp.idx = h->z_idx; rp.mu = h->z_zero_mu; rp.cf = h->d_cf; rp.lut = h->d_lut;
    rp.n_chunks = n; rp.n_sub = h->n_sub_z; rp.h = h->h_z; rp.w = h->w_z; rp.c_y = c.c_z;
    rp.rows_per_sub = c.rows_per_substream; rp.W = c.lanes_per_substream; rp.n_buckets = c.n_buckets;
    rp.y_stride = c.c_z;
    rp.yhat = h->z_scratch; rp.sym_tap = h->z_hwc; rp.yhat_tap = nullptr; rp.status = h->d_status;
    CU_TRY(launch_rans_decode(rp, st));
    CU_TRY(launch_z_hwc_to_planar(h->z_hwc, z_planar_out, n, c.c_z, h->h_z * h->w_z, st));
    if (launches) *launches += 2;
    return UFNVC_OK;
}
}  // namespace

extern "C" int ufnvc_decode_z(ufnvc_handle *h, int n_chunks, const uint8_t *bits_dev, size_t bits_bytes, const uint32_t *sub_off_dev,
                              int16_t *z_dev, void *cuda_stream)
{
    if (!h) return UFNVC_E_INVALID_ARG;
    if (!h->weights_loaded) return fail(h, UFNVC_E_NO_WEIGHTS, "ufnvc_load_weights has not succeeded on this handle");
    if (n_chunks < 1 || n_chunks > h->max_chunks) return fail(h, UFNVC_E_INVALID_ARG, "n_chunks outside [1, max_chunks_per_call]");
    if (!bits_dev || !sub_off_dev || !z_dev) return fail(h, UFNVC_E_INVALID_ARG, "null device pointer");
    if (reinterpret_cast<uintptr_t>(bits_dev) & 3) return fail(h, UFNVC_E_INVALID_ARG, "bits_dev must be 4-byte aligned");
    int launches = 0;
    const int rc = decode_z_impl(h, n_chunks, bits_dev, bits_bytes, sub_off_dev, h->n_sub_z, z_dev, static_cast<cudaStream_t>(cuda_stream),
                                 &launches);
    h->last_launches = launches;
    return rc;
}

extern "C" int ufnvc_chunk_decode_bytes(ufnvc_handle *h, int n_chunks, const uint8_t *bits_dev, size_t bits_bytes,
                                        const uint32_t *sub_off_dev, float *frames_dev, void *cuda_stream)
{
    if (!h) return UFNVC_E_INVALID_ARG;
    if (!h->weights_loaded) return fail(h, UFNVC_E_NO_WEIGHTS, "ufnvc_load_weights has not succeeded on this handle");
    if (n_chunks < 1 || n_chunks > h->max_chunks) return fail(h, UFNVC_E_INVALID_ARG, "n_chunks outside [1, max_chunks_per_call]");
    if (!bits_dev || !sub_off_dev || !frames_dev) return fail(h, UFNVC_E_INVALID_ARG, "null device pointer");
    if (reinterpret_cast<uintptr_t>(bits_dev) & 3) return fail(h, UFNVC_E_INVALID_ARG, "bits_dev must be 4-byte aligned");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int launches = 0;
    if (int rc = decode_z_impl(h, n_chunks, bits_dev, bits_bytes, sub_off_dev, h->n_sub_z + h->n_sub, h->z_planar, st, &launches)) return rc;
    // the y decode ORs into the same status word: keep the z stage's bits by skipping run()'s reset
    h->y_sub_stride = h->n_sub_z + h->n_sub;
    h->keep_status = true;
    const int rc = run(h, n_chunks, h->z_planar, bits_dev, bits_bytes, sub_off_dev, frames_dev, st, nullptr, nullptr, nullptr, false,
                       nullptr, nullptr, nullptr, nullptr, &launches);
    h->y_sub_stride = 0;
    h->keep_status = false;
    return rc;
}

// ---- NEXT-4 (part): GPU rANS encode of r, the mirror of A3 ---------------------------------------------------------
namespace {
// idx + r on the device -> the bit-stream ufnvc_chunk_decode takes (rans_encode.cu); allocates its scratch on first use
int encode_dev_impl(ufnvc_handle *h, int n_chunks, const uint8_t *idx_dev, const int16_t *sym_dev, uint8_t *bits_dev, size_t cap,
                    uint32_t *sub_off_dev, cudaStream_t stream, bool clear_status)
{
    const ufnvc_config &c = h->cfg;
    const LaunchStream st{stream, h->pdl};
    const int G = c.lanes_per_substream / 32;
    if (!h->enc_tmp) {
        const size_t n_sym = size_t(c.rows_per_substream) * h->w * c.c_y;
        const size_t steps = (n_sym + c.lanes_per_substream - 1) / c.lanes_per_substream;
        h->enc_tmp_stride = steps * 32;
        h->enc_stage_stride = (size_t(8) * G + size_t(G) * 132 + 2 * steps * c.lanes_per_substream + 31) / 16 * 16;
        const size_t subs = size_t(h->max_chunks) * h->n_sub;
        void *a = nullptr, *b = nullptr, *d = nullptr;
        if (cudaMalloc(&a, subs * G * h->enc_tmp_stride * 2) != cudaSuccess || cudaMalloc(&b, subs * h->enc_stage_stride) != cudaSuccess ||
            cudaMalloc(&d, subs * 4) != cudaSuccess) {
            cudaFree(a); cudaFree(b); cudaFree(d);
            cudaGetLastError();
            return fail(h, UFNVC_E_OOM, "cudaMalloc failed (encoder scratch)");
        }
        h->allocs.push_back(a); h->allocs.push_back(b); h->allocs.push_back(d);
        h->enc_tmp = static_cast<uint16_t *>(a); h->enc_stage = static_cast<uint8_t *>(b); h->enc_sizes = static_cast<uint32_t *>(d);
    }
    if (clear_status) CU_TRY(cudaMemsetAsync(h->d_status, 0, 4, stream));
    RansEncParams p{};
    p.idx = idx_dev; p.sym = sym_dev; p.cf = h->d_cf;
    p.n_chunks = n_chunks; p.n_sub = h->n_sub; p.h = h->h; p.w = h->w; p.c_y = c.c_y;
    p.rows_per_sub = c.rows_per_substream; p.W = c.lanes_per_substream; p.n_buckets = c.n_buckets;
    p.tmp_words = h->enc_tmp; p.tmp_stride = h->enc_tmp_stride; p.stage = h->enc_stage; p.stage_stride = h->enc_stage_stride;
    p.sizes = h->enc_sizes; p.bits_out = bits_dev; p.cap = cap; p.sub_off = sub_off_dev; p.status = h->d_status;
    CU_TRY(launch_rans_encode(p, st));
    return UFNVC_OK;
}
}  // namespace

extern "C" int ufnvc_encode_chunk_dev(ufnvc_handle *h, int n_chunks, const uint8_t *idx_dev, const int16_t *sym_dev, uint8_t *bits_dev,
                                      size_t cap, uint32_t *sub_off_dev, void *cuda_stream)
{
    if (!h) return UFNVC_E_INVALID_ARG;
    if (n_chunks < 1 || n_chunks > h->max_chunks) return fail(h, UFNVC_E_INVALID_ARG, "n_chunks outside [1, max_chunks_per_call]");
    if (!idx_dev || !sym_dev || !bits_dev || !sub_off_dev) return fail(h, UFNVC_E_INVALID_ARG, "null device pointer");
    if (reinterpret_cast<uintptr_t>(bits_dev) & 3) return fail(h, UFNVC_E_INVALID_ARG, "bits_dev must be 4-byte aligned");
    const int rc = encode_dev_impl(h, n_chunks, idx_dev, sym_dev, bits_dev, cap, sub_off_dev, static_cast<cudaStream_t>(cuda_stream), true);
    h->last_launches = 2;
    return rc;
}

extern "C" int ufnvc_entropy_params(ufnvc_handle *h, int n_chunks, const int16_t *z_dev, float *mu_dev, float *lnscale_dev,
                                    uint8_t *idx_dev, void *cuda_stream)
{
    if (!h) return UFNVC_E_INVALID_ARG;
    if (!h->weights_loaded) return fail(h, UFNVC_E_NO_WEIGHTS, "ufnvc_load_weights has not succeeded on this handle");
    if (n_chunks < 1 || n_chunks > h->max_chunks || !z_dev) return fail(h, UFNVC_E_INVALID_ARG, "bad n_chunks or null z_dev");
    return run(h, n_chunks, z_dev, nullptr, 0, nullptr, nullptr, static_cast<cudaStream_t>(cuda_stream), nullptr, nullptr, nullptr, true,
               mu_dev, lnscale_dev, idx_dev, nullptr, nullptr);
}

extern "C" int ufnvc_launches_per_call(const ufnvc_handle *h, int n_chunks)
{
    if (!h || n_chunks < 1) return UFNVC_E_INVALID_ARG;
    // kernels counted by the last decode on this handle (the count does not depend on n_chunks); before any decode, the
    // count of the default path: 4 hyper (hybrid head) + rANS + A5 + (depthwise + fused MLP) per trunk block + 4 stages
    if (h->last_launches > 0) return h->last_launches;
    return 4 + 1 + 1 + 2 * h->cfg.n_trunk_blocks + 4;
}

extern "C" int ufnvc_chunk_decode_profiled(ufnvc_handle *h, int n_chunks, const int16_t *z_dev, const uint8_t *bits_dev,
                                           size_t bits_bytes, const uint32_t *sub_off_dev, float *frames_dev, void *cuda_stream,
                                           int detail, float *us_out_host)
{
    if (int rc = check_call(h, n_chunks, z_dev, bits_dev, sub_off_dev)) return rc;
    if (!frames_dev || !us_out_host) return fail(h, UFNVC_E_INVALID_ARG, "null frames_dev / us_out_host");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (!h->ev_made) {
        for (auto &e : h->ev) CU_TRY(cudaEventCreate(&e));
        h->ev_made = true;
    }
    if (h->ev_dw.size() < size_t(2 * h->cfg.n_trunk_blocks)) {
        const size_t old = h->ev_dw.size();
        h->ev_dw.resize(size_t(2 * h->cfg.n_trunk_blocks));
        for (size_t i = old; i < h->ev_dw.size(); ++i) CU_TRY(cudaEventCreate(&h->ev_dw[i]));
    }
    Stage sg{h->ev, 0, (detail && !h->ev_dw.empty()) ? h->ev_dw.data() : nullptr};
    if (int rc = run(h, n_chunks, z_dev, bits_dev, bits_bytes, sub_off_dev, frames_dev, st, nullptr, nullptr, nullptr, false, nullptr,
                     nullptr, nullptr, &sg, nullptr))
        return rc;
    CU_TRY(cudaStreamSynchronize(st));
    // events: 0 start, 1 after A1+A2, 2 after A3+A4, 3 after A5, 4 after trunk, 5 after A8, 6 after A9, 7 after the context generation
    {
        float ms = 0.f;
        CU_TRY(cudaEventElapsedTime(&ms, h->ev[6], h->ev[7]));
        us_out_host[7] = ms * 1000.f;
    }
    for (int i = 0; i < 6; ++i) {
        float ms = 0.f;
        CU_TRY(cudaEventElapsedTime(&ms, h->ev[i], h->ev[i + 1]));
        us_out_host[i] = ms * 1000.f;
    }
    // us_out_host[6] = A6 alone: the sum over the trunk blocks of (event after the depthwise launch - event before it)
    float dw_us = 0.f;
    for (int k = 0; detail && k < h->cfg.n_trunk_blocks; ++k) {
        float ms = 0.f;
        CU_TRY(cudaEventElapsedTime(&ms, h->ev_dw[2 * k + 1], h->ev_dw[2 * k]));
        dw_us += ms * 1000.f;
    }
    us_out_host[6] = dw_us;
    return UFNVC_OK;
}

// ---- NEXT-2a (R23): the temporal context state ------------------------------------------------------------------------
namespace {
int ctx_call_ok(ufnvc_handle *h, int n_chunks)
{
    if (!h) return UFNVC_E_INVALID_ARG;
    if (!h->has_ctx) return fail(h, UFNVC_E_BAD_CONFIG, "this handle has no temporal context (n_ctx_blocks == 0)");
    if (!h->weights_loaded) return fail(h, UFNVC_E_NO_WEIGHTS, "ufnvc_load_weights has not succeeded on this handle");
    if (n_chunks < 1 || n_chunks > h->max_chunks) return fail(h, UFNVC_E_INVALID_ARG, "n_chunks outside [1, max_chunks_per_call]");
    return UFNVC_OK;
}
int ctx_refresh_prior(ufnvc_handle *h, int n, cudaStream_t stream)
{
    const ufnvc_config &c = h->cfg;
    const LaunchStream st{stream, false};          // follows a copy / memset node: plain stream order
    CU_TRY(launch_ctx_prior(h->yhat + c.c_y, h->c_cat, c.c_trunk, h->ctx_prior_w, h->ctx_prior_b, h->ctx_q, n, h->h, h->w, h->h_z, h->w_z,
                            c.c_hyper, st));
    return UFNVC_OK;
}
}  // namespace

extern "C" int ufnvc_reset_context(ufnvc_handle *h, int n_chunks, void *cuda_stream)
{
    if (int rc = ctx_call_ok(h, n_chunks)) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const ufnvc_config &c = h->cfg;
    const size_t rows = size_t(n_chunks) * h->h * h->w;
    CU_TRY(cudaMemset2DAsync(h->yhat + c.c_y, size_t(h->c_cat) * 2, 0, size_t(c.c_trunk) * 2, rows, st));
    return ctx_refresh_prior(h, n_chunks, st);      // q of the zero context is ReLU(b_p), not zero
}

extern "C" int ufnvc_get_context(ufnvc_handle *h, int n_chunks, uint16_t *ctx_dev, void *cuda_stream)
{
    if (int rc = ctx_call_ok(h, n_chunks)) return rc;
    if (!ctx_dev) return fail(h, UFNVC_E_INVALID_ARG, "null ctx_dev");
    const ufnvc_config &c = h->cfg;
    const size_t rows = size_t(n_chunks) * h->h * h->w;
    CU_TRY(cudaMemcpy2DAsync(ctx_dev, size_t(c.c_trunk) * 2, h->yhat + c.c_y, size_t(h->c_cat) * 2, size_t(c.c_trunk) * 2, rows,
                             cudaMemcpyDeviceToDevice, static_cast<cudaStream_t>(cuda_stream)));
    return UFNVC_OK;
}

extern "C" int ufnvc_set_context(ufnvc_handle *h, int n_chunks, const uint16_t *ctx_dev, void *cuda_stream)
{
    if (int rc = ctx_call_ok(h, n_chunks)) return rc;
    if (!ctx_dev) return fail(h, UFNVC_E_INVALID_ARG, "null ctx_dev");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const ufnvc_config &c = h->cfg;
    const size_t rows = size_t(n_chunks) * h->h * h->w;
    CU_TRY(cudaMemcpy2DAsync(h->yhat + c.c_y, size_t(h->c_cat) * 2, ctx_dev, size_t(c.c_trunk) * 2, size_t(c.c_trunk) * 2, rows,
                             cudaMemcpyDeviceToDevice, st));
    return ctx_refresh_prior(h, n_chunks, st);
}

// ---- NEXT-4 (R24): chunk ENCODE, frames -> bytes --------------------------------------------------------------------------
// E1 patch gather + 1x1 embedding (space-to-depth x2 store) -> E2 fold over the T frames -> E3 + context -> E4 DC blocks ->
// E5 latent head (fp32) -> E6 hyper-encoder (z) -> the decoder's prior net on z (A1 + A2) -> E8 quantiser -> GPU rANS encoder.
extern "C" int ufnvc_chunk_encode(ufnvc_handle *h, int n_chunks, const float *frames_dev, uint8_t *bits_dev, size_t cap,
                                  uint32_t *sub_off_dev, int16_t *z_dev, const ufnvc_enc_taps *taps, void *cuda_stream)
{
    if (!h) return UFNVC_E_INVALID_ARG;
    if (!h->has_enc) return fail(h, UFNVC_E_BAD_CONFIG, "this handle has no encoder (n_enc_blocks == 0)");
    if (!h->weights_loaded) return fail(h, UFNVC_E_NO_WEIGHTS, "ufnvc_load_weights has not succeeded on this handle");
    if (n_chunks < 1 || n_chunks > h->max_chunks) return fail(h, UFNVC_E_INVALID_ARG, "n_chunks outside [1, max_chunks_per_call]");
    if (!frames_dev || !bits_dev || !sub_off_dev || !z_dev) return fail(h, UFNVC_E_INVALID_ARG, "null device pointer");
    if (reinterpret_cast<uintptr_t>(bits_dev) & 3) return fail(h, UFNVC_E_INVALID_ARG, "bits_dev must be 4-byte aligned");
    if (taps && taps->struct_size != sizeof(ufnvc_enc_taps)) return fail(h, UFNVC_E_INVALID_ARG, "ufnvc_enc_taps.struct_size mismatch");
    const ufnvc_config &c = h->cfg;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const LaunchStream st{stream, h->pdl};
    const int n = n_chunks, T = c.T, Ct = c.c_trunk, P = h->h * h->w, Pz = h->h_z * h->w_z;
    int launches = 0;
    // one memset for the status word and the encoder blocks' tile counters (same block of words the decode call clears)
    {
        const size_t words = h->tail_fill ? 4 + size_t(c.n_trunk_blocks + c.n_enc_blocks) * h->trunk_sync_stride : 4;
        CU_TRY(cudaMemsetAsync(h->zero_block, 0, words * 4, stream));
    }
    // E1: 8x8 patches of every frame, then the 1x1 embedding whose epilogue stores space-to-depth x2 (ready for the fold)
    CU_TRY(launch_enc_patchify(frames_dev, h->p8, n * T, c.height, c.width, 2 * h->h, 2 * h->w, st));
    ++launches;
    {
        ConvProblem pr{h->p8, n * T, 2 * h->h, 2 * h->w, 1};
        EpiParams E{EPI_NHWC, ACT_NONE, h->s2, nullptr, Ct, 0, (long long)P * 4 * Ct, 0, 0, 0};
        E.unps2 = 1;
        CU_TRY(conv(h, h->enc_patch, pr, h->am_p8, E, st, &launches));
    }
    // E2: fold over the T frames (tap t = frame t of the chunk), 4 c_trunk channels each
    {
        ConvProblem pr{h->s2, n, h->h, h->w, 1, true};
        EpiParams E{EPI_NHWC, ACT_NONE, h->ca, nullptr, Ct, 0, (long long)P * Ct, 0, 0, 0};
        CU_TRY(conv(h, h->enc_fold, pr, h->am_s2, E, st, &launches));
    }
    // E3: + 1x1 conv of the temporal context C_i, read in place from the [y ; C] buffer
    if (h->has_ctx) {
        ConvProblem pr{h->yhat + c.c_y, n, h->h, h->w, 1};
        EpiParams E{EPI_NHWC, ACT_NONE, h->ca, h->ca, Ct, 0, (long long)P * Ct, 0, 0, 0};
        CU_TRY(conv(h, h->enc_ctx, pr, h->am_cin, E, st, &launches));
    }
    // E4: the chunk encoder's DC blocks, on the depthwise + fused MLP kernels of the trunk (one image per chunk)
    for (int k = 0; k < c.n_enc_blocks; ++k) {
        const ufnvc_handle::TrunkBlock &tb = h->enc_blocks[k];
        uint32_t *sync_k = h->trunk_sync + size_t(c.n_trunk_blocks + k) * h->trunk_sync_stride;
        const bool mlp_counts = trunk_counts_tiles((long long)n * P, h->use_pair_trunk) && h->tail_fill;
        CU_TRY(launch_dwconv3x3_tma(h->tm_dw_ctx, h->cb, tb.dw_w, tb.dw_b, n, h->h, h->w, Ct, h->num_sms, st, h->tail_fill ? sync_k : nullptr,
                                    (k > 0 && mlp_counts) ? sync_k - h->trunk_sync_stride + 1 : nullptr));
        CU_TRY(launch_trunk_mlp(tb.fused, tb.pw1, tb.pw2, h->ca, h->ca, (long long)n * P, h->num_sms, h->use_pair_trunk, st,
                                mlp_counts ? sync_k + 1 : nullptr, h->use_quad_clusters));
        launches += 2;
    }
    // E5: latent head, fp32 out
    {
        ConvProblem pr{h->ca, n, h->h, h->w, 1};
        EpiParams E{EPI_NHWC, ACT_NONE, h->ey, nullptr, c.c_y, 0, (long long)P * c.c_y, 0, 0, 0};
        E.out_f32 = 1;
        CU_TRY(conv(h, h->enc_y, pr, h->am_ca, E, st, &launches));
    }
    // E6: hyper-encoder -> z (int16, planar: what A1 reads), then the decoder's own prior net on it
    CU_TRY(launch_hyper_encoder(h->ey, h->henc_w0, h->henc_b0, h->henc_w1, h->henc_b1, h->henc_a, h->ez, taps ? taps->zf : nullptr, n, h->h, h->w,
                                h->h_z, h->w_z, c.c_y, c.c_hyper, c.c_z, st));
    launches += 2;
    CU_TRY(cudaMemcpyAsync(z_dev, h->ez, size_t(n) * Pz * c.c_z * 2, cudaMemcpyDeviceToDevice, stream));
    {
        h->keep_status = true;                 // run() must not clear what this call's memset cleared (it would also re-clear counters)
        const int rc = run(h, n, h->ez, nullptr, 0, nullptr, nullptr, stream, nullptr, nullptr, nullptr, true, nullptr, nullptr, nullptr, nullptr,
                           &launches);
        h->keep_status = false;
        if (rc) return rc;
    }
    // E8: r = round(y - mu), then the mirror of A3
    const size_t ne = size_t(n) * P * c.c_y;
    CU_TRY(launch_enc_quantise(h->ey, h->mu, h->esym, (long long)ne, st));
    ++launches;
    if (taps) {
        if (taps->y) CU_TRY(cudaMemcpyAsync(taps->y, h->ey, ne * 4, cudaMemcpyDeviceToDevice, stream));
        if (taps->sym) CU_TRY(cudaMemcpyAsync(taps->sym, h->esym, ne * 2, cudaMemcpyDeviceToDevice, stream));
        if (taps->mu) CU_TRY(cudaMemcpyAsync(taps->mu, h->mu, ne * 4, cudaMemcpyDeviceToDevice, stream));
        if (taps->idx) CU_TRY(cudaMemcpyAsync(taps->idx, h->idx, ne, cudaMemcpyDeviceToDevice, stream));
    }
    if (int rc = encode_dev_impl(h, n, h->idx, h->esym, bits_dev, cap, sub_off_dev, stream, false)) return rc;
    h->last_launches = launches + 2;
    return UFNVC_OK;
}
