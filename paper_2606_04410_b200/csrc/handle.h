// The opaque handle behind include/ufnvc.h: config, geometry, device weights, tables, workspace.
#pragma once
#include <map>
#include <string>
#include <vector>

#include "ufnvc_internal.h"

struct ufnvc_handle {
    ufnvc_config cfg{};
    // geometry (SURVEY.md section 8 notation)
    int H = 0, W = 0, h = 0, w = 0, h_z = 0, w_z = 0, n_sub = 0;
    int num_sms = 0;
    int max_chunks = 1;
    bool weights_loaded = false;
    int last_launches = 0;               // kernels enqueued by the last decode call (ufnvc_launches_per_call)
    // code-path switches, all derived from ufnvc_config.debug_flags at create (include/ufnvc.h UFNVC_DBG_*; 0 = defaults)
    bool use_pair_conv = true;           // CTA-pair halo conv for A8 (else single-CTA)
    bool use_pair_trunk = true;          // CTA-pair fused MLP kernel (else single-CTA)
    bool use_fused_trunk = true;         // fused MLP kernel (else two 1x1 conv launches per block)
    bool force_generic = false;          // CUDA-core convs everywhere (cross-check)
    bool pdl = true;                     // programmatic dependent launch along the kernel chain
    bool use_final_is = true;            // A9 input-stationary kernel
    bool use_dw_tma = true;              // A6 TMA-staged kernel
    bool use_transposed_tiles = true;    // CTA-pair halo conv: 8 x 16 tiles where they pad the image less
    bool use_quad_clusters = true;       // fused MLP kernel: clusters of two CTA pairs sharing the weight tiles by multicast
    std::string err;

    // entropy tables (O3)
    std::vector<uint32_t> cdf32;         // [nb][256], host copy
    uint32_t *d_cf = nullptr;             // [nb][256]: c[pos] | freq[pos] << 16
    uint32_t *d_lut = nullptr;
    uint32_t *d_status = nullptr;

    // layers
    ufnvc::HyperLayer hyper[3];
    // hybrid head (R12): tensor-core evaluation of the last hyper conv + exact fp64 re-evaluation near bucket edges
    bool hybrid_head = false;
    // a-priori bound on |tensor-core ln sigma - fp64 ln sigma| = head_kappa * |w row|_2 * |x patch|_2 (decode.cu); elements
    // closer than that to a bucket edge are re-decided in fp64
    double head_kappa = 0.0;
    float *head_wnorm = nullptr;         // [2 c_y 16] |w row|_2 per packed head column
    float *xnorm2 = nullptr;             // [n][h_z][w_z] sum over channels of hx2^2
    ufnvc::ConvLayer head_tc;
    double *head_fix_w = nullptr, *head_fix_b = nullptr;   // [c_y*16][9][c_hyper], [c_y*16] (scale half)
    ufnvc::bf16 *xs = nullptr;           // [n][h_z][w_z][2*c_hyper]: bf16 hi | mid split of the fp64 hx2
    uint32_t *fix_list = nullptr, *fix_count = nullptr;
    ufnvc::ConvLayer xframe;
    ufnvc::ConvLayer mu_net[3];          // mu_steps == 4: 3x3 convs [y so far ; mu0] -> mu^k, k = 1..3 (R21)
    struct TrunkBlock {
        float *dw_w = nullptr, *dw_b = nullptr;   // [9][C], [C] fp32
        ufnvc::ConvLayer pw1, pw2;
        ufnvc::TrunkMaps fused;                   // TMA maps of the fused MLP kernel (per n_chunks: rows = n*T*P)
    };
    std::vector<TrunkBlock> trunk;
    ufnvc::ConvLayer dec[4];             // groups = T
    // temporal chunk context (NEXT-2a, R23).  The state C_i lives in the context block of the [y ; C] buffer
    // (`yhat`, c_cat = c_y + c_trunk channels per pixel) that the cross-frame unfold reads; ctx_q is its prior branch
    // q = ReLU(W_p pool4(C_i) + b_p) in fp64, recomputed whenever the state changes.
    bool has_ctx = false;
    int c_cat = 0;                       // channels per pixel of `yhat`: c_y, or c_y + c_trunk with a context
    ufnvc::ConvLayer ctx_fold, ctx_out;  // 1x1: T c_trunk -> c_trunk (taps = T images), c_trunk -> c_trunk
    std::vector<TrunkBlock> ctx_blocks;
    double *ctx_prior_w = nullptr, *ctx_prior_b = nullptr;   // [c_trunk][c_hyper] (k-major), [c_hyper]
    double *ctx_q = nullptr;             // [n][h_z][w_z][c_hyper]
    ufnvc::bf16 *ca = nullptr, *cb = nullptr;   // [n][h][w][c_trunk] ping-pong of the context generation
    CUtensorMap tm_dw_ctx;               // ca as the depthwise kernel reads it
    bool dw_ctx_ok = false;
    // chunk encoder (NEXT-4, R24): E1 patch embedding, E2 fold over frames, E3 context, E4 DC blocks (on ca / cb),
    // E5 latent head, E6 hyper-encoder, E8 quantiser; then the GPU rANS encoder
    bool has_enc = false;
    ufnvc::ConvLayer enc_patch, enc_fold, enc_ctx, enc_y;
    std::vector<TrunkBlock> enc_blocks;
    float *henc_w0 = nullptr, *henc_b0 = nullptr, *henc_w1 = nullptr, *henc_b1 = nullptr;   // fp32 [16 c_y][c_h], [c_h], [9][c_h][c_z], [c_z]
    ufnvc::bf16 *p8 = nullptr, *s2 = nullptr;   // [n T][H/8][W/8][192] patches; [n T][h][w][4 c_trunk] embedded + space-to-depth x2
    float *ey = nullptr, *henc_a = nullptr;     // [n][h][w][c_y] unquantised latent; [n][h_z][w_z][c_hyper]
    int16_t *esym = nullptr, *ez = nullptr;     // [n][h][w][c_y] residual; [n][c_z][h_z][w_z] hyper-latent

    // workspace (sized for max_chunks)
    double *hx1 = nullptr, *hx2 = nullptr;
    float *mu = nullptr, *lnscale = nullptr;
    uint8_t *idx = nullptr;
    ufnvc::bf16 *yhat = nullptr, *fa = nullptr, *fb = nullptr, *hidden = nullptr;
    ufnvc::bf16 *stage[3] = {nullptr, nullptr, nullptr};
    ufnvc::bf16 *ymu[2] = {nullptr, nullptr};   // mu_steps == 4: [n][h][w][2 c_y] = y decoded so far | mu0, ping-pong
    int16_t *sym = nullptr;                     // mu_steps == 4: decoded residual r, [n][h][w][c_y]
    // NEXT-3 (R22): the hyper-latent's own entropy decode (bytes-only entry points)
    int n_sub_z = 0;
    int y_sub_stride = 0;                       // > 0 while a bytes-only call runs: offset-table entries per chunk
    bool keep_status = false;                   // bytes-only call: the y decode must not clear the z decode's status bits
    bool z_prior_loaded = false;
    std::vector<uint8_t> z_idx_c;               // [c_z] bucket index of each channel's prior (host copy)
    uint8_t *z_idx = nullptr;                   // [n][h_z][w_z][c_z]: z_idx_c broadcast, what the rANS kernel reads
    float *z_zero_mu = nullptr;                 // [n][h_z][w_z][c_z] zeros (the prior is zero-mean)
    ufnvc::bf16 *z_scratch = nullptr;           // the kernel's bf16 "y" output, unused for z
    int16_t *z_hwc = nullptr, *z_planar = nullptr;

    // TMA descriptors of the activation tensors the tcgen05 convs read, built once at create (workspace is fixed)
    struct ActMap {
        CUtensorMap tm;
        int tile_h = 0, tile_w = 0;
        bool flat = false;               // 1x1 convs: all pixels of all images as one [rows][128] matrix
        bool ok = false;
        CUtensorMap tm_halo;             // 3x3 convs: box {64, 10, 18}: a 16 x 8 pixel tile plus halo (conv_halo_kernel)
        bool halo_ok = false;
        CUtensorMap tm_halo_t;           // the same with the image's y as map dimension 1 (CTA-pair kernel), when that pads to fewer tiles
        bool halo_t = false;
    };
    ufnvc::FinalMaps final_is;           // A9 input-stationary kernel
    CUtensorMap tm_dw;                   // fa as the depthwise kernel reads it: box {64 ch, 10, 10}
    bool dw_tma_ok = false;
    // per trunk block: [0] = the depthwise kernel's dynamic tile counter, [1 ..] = one completion counter per 128-pixel tile of
    // the trunk MLP kernel (8 epilogue warps each); zeroed at the start of every call (tail filling)
    uint32_t *trunk_sync = nullptr;
    uint32_t *zero_block = nullptr;      // [0] = status word, [1] = fix_count, [4 ..] = trunk_sync: cleared by one memset per call
    size_t zero_words = 0;
    size_t trunk_sync_stride = 0;
    bool tail_fill = true;
    ActMap am_xs, am_yhat, am_fa, am_fb, am_hidden, am_stage[3], am_ymu[2], am_ca;
    ActMap am_p8, am_s2, am_cin;         // encoder (R24); am_cin: the context block of the [y ; C] buffer as a conv input

    // GPU rANS encoder scratch (NEXT-4), allocated by the first ufnvc_encode_chunk_dev call
    uint16_t *enc_tmp = nullptr;
    uint8_t *enc_stage = nullptr;
    uint32_t *enc_sizes = nullptr;
    size_t enc_tmp_stride = 0, enc_stage_stride = 0;
    // ufnvc_encode_chunk_dev_static: device address of encode_static.cu's file-scope scratch array on this handle's device
    // (cudaGetSymbolAddress at create; nullptr if that failed)
    void *static_scratch = nullptr;

    std::vector<void *> allocs;          // workspace and tables, freed at destroy
    std::vector<void *> weight_allocs;   // what ufnvc_load_weights uploaded; freed by the next load and at destroy
    cudaEvent_t ev[9] = {};
    std::vector<cudaEvent_t> ev_dw;      // profiled call: before / after every depthwise launch
    bool ev_made = false;
};

namespace ufnvc {
int fail(ufnvc_handle *h, int code, const std::string &msg);
int load_weights_impl(ufnvc_handle *h, const void *blob, size_t bytes);
}  // namespace ufnvc
