// Internal declarations of libufnvc (not part of the ABI).  sm_100a only.
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdlib>
#include <string>
#include <vector>

#include "../../include/ufnvc.h"

namespace ufnvc {

typedef __nv_bfloat16 bf16;

// ---- epilogue description shared by the CUDA-core and the tcgen05 conv kernels -------------------------------
enum EpiMode : int {
    EPI_NHWC = 0,   // out[img][split][pix][n % n_split]  (bf16), optional residual with the same indexing
    EPI_PS2 = 1,    // pixel-shuffle x2 (R14): packed column n' = (2i+j)*C_o + c -> out[img][2y+i][2x+j][c] (bf16)
    EPI_FINAL = 2,  // EPI_PS2 + clamp [0,1] + crop + planar fp32 store out[img][c][Y][X]  (A9)
    EPI_HEAD = 3,   // hyper head (A2): pixel-shuffle x4 + crop; mu half -> fp32, scale half -> clamp, bucket, edge flag
    EPI_MU = 4      // progressive means (R21): column n = latent channel; y = r + mu^k on partition k, old y elsewhere
};
enum Act : int { ACT_NONE = 0, ACT_GELU = 1 };

struct EpiParams {
    int mode, act;
    void *out;
    const bf16 *residual;    // EPI_NHWC only; may alias out
    int n_split;             // EPI_NHWC: channels per output group (xframe: c_trunk, else N)
    long long split_stride;  // EPI_NHWC: elements between output groups
    long long img_stride;    // output elements per input image
    int c_o;                 // EPI_PS2/FINAL: channels after the shuffle (N = 4*c_o)
    int out_h, out_w;        // EPI_FINAL: crop (height, width)
    // EPI_HEAD: packed column n' = (s*16 + 4i+j)*c_y + c2 of z-pixel (zy, zx) -> latent (4zy+i, 4zx+j), channel c2
    float *mu, *lnscale;     // [n][lat_h][lat_w][c_y]
    uint8_t *idx;
    uint32_t *fix_list, *fix_count;   // elements whose tensor-core ln sigma may be on the wrong side of a bucket edge
    int c_y, lat_h, lat_w, n_buckets;
    float ln_lo, ln_hi, t_scale;      // t = (u - ln_lo) * t_scale + 0.5
    // element (z-pixel m, packed column n') is flagged when |t - round(t)| < kappa_t * wnorm[n'] * sqrt(sum of xnorm2 over the
    // 3x3 neighbourhood of m): the a-priori bound on the tensor-core value's error, in bucket units (decode.cu)
    const float *wnorm;               // [n_pad]: L2 norm of packed weight row n' over its 9 * c_hyper taps
    const float *xnorm2;              // [n][h_z][w_z][xnorm_parts]: shares of the sum over channels of the squared layer-2 activation
    int xnorm_parts;
    float kappa_t;
    // EPI_MU (uses c_y), mu^k = acc + bias.  The conv input is [r so far | mu used so far | mu0 | pad] (bf16, in_stride
    // channels).  mu_last == 0: out has the same layout: r and mu blocks updated on partition mu_step.
    // mu_last == 1: out = dense y = r + mu, [pix][out_stride] (what A5 reads).
    const int16_t *sym;      // [pix][c_y] decoded residual r
    const bf16 *y_in;        // the conv's own input
    int in_stride, out_stride, mu_step, mu_last;
    float *mu_tap, *yhat_tap;   // optional fp32 [pix][c_y], written on partition mu_step only
    int unps2;               // EPI_NHWC: 1 = space-to-depth x2 store (R24 E1 -> E2): pixel (y, x), column n ->
                             // out[img][y / 2][x / 2][(2 (y % 2) + x % 2) n_split + n]
    int out_f32;             // EPI_NHWC: 1 = `out` is fp32 (the unquantised latent y, R24 E5)
    int pix_stride;          // EPI_NHWC: elements between pixels of a group; 0 = n_split (dense).  > n_split: the conv writes a
                             // channel block of a wider tensor (context generation -> [y ; C] buffer, R23)
};

// R21: partition of latent element (channel c, row y, column x): four channel groups x the four positions of a 2x2 cell
__host__ __device__ inline int mu_partition(int c, int y, int x, int c_y) { return (2 * (y & 1) + (x & 1) + (4 * c) / c_y) & 3; }

// One conv layer as the kernels consume it.  Weights are K-major ("[n][k]", k = c_in contiguous) per tap and
// per weight group: w[group][tap][n_pad][c_in] bf16; bias[group][n_pad] fp32.  For EPI_PS2/FINAL layers the
// rows are permuted at load time so that packed row n' = (2i+j)*C_o + c holds canonical row 4c + 2i + j.
struct ConvLayer {
    int c_in = 0, n = 0, n_pad = 0, taps = 1, groups = 1;
    bf16 *w = nullptr;
    float *bias = nullptr;
    std::vector<float> bias_host;   // host copy of bias (group 0 .. groups-1, n_pad each): kernels that take biases by value
    bool use_tc = false;     // tcgen05 path eligible (c_in % 64 == 0, n_pad % 16 == 0)
    CUtensorMap tmap_w;      // 3-D {c_in, n_pad, groups*taps}, box {64, block_n, 1}, 128B swizzle
    CUtensorMap tmap_w_half; // same tensor, box {64, block_n / 2, 1}: one CTA's half of a weight tile (CTA-pair kernel)
    bool has_half_map = false;
    int block_n = 0;
};

struct ConvProblem {
    const bf16 *in;          // [n_img][H][W][c_in] bf16 NHWC
    int n_img, H, W;
    int imgs_per_group_cycle; // weight group of image i = (groups == 1) ? 0 : i % groups
    bool taps_are_images = false;   // 1x1 "fold" over T stacked images (R23): tap t reads image img * taps + t of `in` (n_img output images)
    bool reverse = false;           // CTA-pair halo kernel: walk the schedule backwards -- the tiles the producer kernel wrote last
                                    // (still in L2) are read first
};

// ---- kernels (each .cu exposes host launchers; all enqueue on `st` and return cudaGetLastError()) -------------
// The stream a launcher enqueues on plus the per-handle launch mode.  pdl: launch with programmatic stream serialization
// (see pdl_grid_sync in tc_ptx.cuh); off = plain stream order (ufnvc_config.debug_flags & UFNVC_DBG_NO_PDL, for A/B timing).
struct LaunchStream {
    cudaStream_t s;
    bool pdl;
    operator cudaStream_t() const { return s; }
};
// Launch with an optional cluster of cluster_x CTAs and, when st.pdl, programmatic stream serialization.
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kern)(KArgs...), unsigned grid, unsigned block, size_t smem, LaunchStream st, int cluster_x, Args &&...args)
{
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = smem; cfg.stream = st.s;
    cudaLaunchAttribute attr[2];
    unsigned n = 0;
    if (cluster_x > 1) {
        attr[n].id = cudaLaunchAttributeClusterDimension;
        attr[n].val.clusterDim.x = unsigned(cluster_x); attr[n].val.clusterDim.y = 1; attr[n].val.clusterDim.z = 1;
        ++n;
    }
    if (st.pdl) {
        attr[n].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[n].val.programmaticStreamSerializationAllowed = 1;
        ++n;
    }
    cfg.attrs = attr; cfg.numAttrs = n;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl_grid(void (*kern)(KArgs...), dim3 grid, unsigned block, LaunchStream st, Args &&...args)   // 3-D grid, no dynamic smem
{
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid; cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = 0; cfg.stream = st.s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = st.pdl ? 1u : 0u;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl_grid_smem(void (*kern)(KArgs...), dim3 grid, unsigned block, size_t smem, LaunchStream st, Args &&...args)   // 3-D grid + dynamic smem
{
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid; cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = smem; cfg.stream = st.s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = st.pdl ? 1u : 0u;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) for every kernel of a translation unit that needs more than 48 KB, on the
// CURRENT device.  Function attributes are per device: ufnvc_create calls all of these for the device the handle lives on, so
// the launchers hold no "already configured" state (a second handle on another GPU of the same process configures that GPU).
cudaError_t configure_rans_kernels();
cudaError_t configure_hyper_kernels();
cudaError_t configure_depthwise_kernels();
cudaError_t configure_conv_tc_kernels();
cudaError_t configure_trunk_kernels();
cudaError_t configure_final_kernels();

cudaError_t launch_conv_generic(const ConvLayer &L, const ConvProblem &P, const EpiParams &E, LaunchStream st);
cudaError_t launch_dwconv3x3(const bf16 *in, bf16 *out, const float *w9c, const float *bias, int n_img, int H, int W,
                             int C, LaunchStream st);

// progressive means, step 0 (R21): ymu0 = [partition 0 ? r : 0 | partition 0 ? mu0 : 0 | mu0 | pad], ymu1's mu0 block
cudaError_t launch_mu_prep(const int16_t *sym, const float *mu0, bf16 *ymu0, bf16 *ymu1, int n_img, int H, int W, int c_y, int stride,
                           LaunchStream st);

cudaError_t launch_dwconv3x3_tma(const CUtensorMap &tm_in, bf16 *out, const float *w9c, const float *bias, int n_img, int H, int W,
                                 int C, int num_sms, LaunchStream st, uint32_t *sched = nullptr, const uint32_t *dep_flags = nullptr);   // tm_in: NHWC map of `in` with box {64, 10, 10, 1}

// fp64 hyper-decoder (A1 + A2), R12: the scale decision is taken in double on both sides.
struct HyperLayer {
    int c_in = 0, n = 0;
    double *w = nullptr;     // [9][c_in][n]
    double *bias = nullptr;  // [n]
};
// layers 0 / 1 of the hyper-decoder (O1) in fp64, one launch each.  in: the int16 hyper-latent, planar [n][c_z][pz]
// (in_is_z), or the previous layer's NHWC fp64 output.  Optional (layer 1): addend [M][n] added AFTER the ReLU -- the context
// branch q of the prior input s = x2 + q (R23); xs = 2-term bf16 split hi | mid of the result; xnorm2[M][hyper_xnorm_parts]
// = per-pixel shares of sum_c v^2.
cudaError_t launch_hyper_conv(const HyperLayer &L, const void *in, bool in_is_z, double *out, int n_img, int hz, int wz, LaunchStream st,
                              bf16 *xs = nullptr, float *xnorm2 = nullptr, const double *addend = nullptr);
int hyper_xnorm_parts(const HyperLayer &L);
// q = ReLU(W_p pool4(C) + b_p) in fp64 from the bf16 context block of the [y ; C] buffer (R23): ctx [n][h][w][stride] (channel
// block already offset), w_p [c_ctx][c_h] (k-major), q [n][h_z][w_z][c_h]
cudaError_t launch_ctx_prior(const bf16 *ctx, int stride, int c_ctx, const double *w_p, const double *b_p, double *q, int n_img, int h, int w,
                             int hz, int wz, int c_h, LaunchStream st);
struct HeadParams {
    int c_y, h, w, n_buckets;
    double ln_lo, ln_hi;
    float *mu, *lnscale;     // [n][h][w][c_y], lnscale may be null
    uint8_t *idx;
};
// hybrid head helpers (hyper.cu)
cudaError_t launch_hyper_fix(const uint32_t *list, const uint32_t *count, const double *x2, const double *fix_w, const double *fix_b,
                             int c_h, int hz, int wz, const HeadParams &hp, int num_sms, LaunchStream st);
cudaError_t launch_hyper_head(const HyperLayer &L, const double *in, int n_img, int hz, int wz, const HeadParams &hp,
                              LaunchStream st);

// rANS decode + dequantisation (A3 + A4)
struct RansParams {
    const uint8_t *bits;
    size_t bits_bytes;
    const uint32_t *sub_off;  // substream s of chunk c: entries [c * sub_stride + sub_first + s] and the next one
    int sub_stride, sub_first;   // (n_sub, 0) for the y-only container; (n_sub_z + n_sub, 0 | n_sub_z) for the bytes-only one
    const uint8_t *idx;       // [n][h][w][c_y]
    const float *mu;
    const uint32_t *cf;       // [nb][256]: c[pos] | freq[pos] << 16
    const uint32_t *lut;      // [nb][kLutBuckets]: search accelerator entry of bin slot >> kLutShift (tables.cu)
    int n_chunks, n_sub, h, w, c_y, rows_per_sub, W, n_buckets;
    int y_stride;             // elements between pixels of yhat (c_y = dense; c_y + C_c when y shares a buffer with the context, R23)
    bf16 *yhat;               // [n][h][w][y_stride], channels [0, c_y)
    int16_t *sym_tap;         // optional
    float *yhat_tap;          // optional
    uint32_t *status;         // device word, OR-ed
};
cudaError_t launch_rans_decode(const RansParams &p, LaunchStream st);

// GPU rANS encode (rans_encode.cu), mirror of the decoder: same geometry fields
struct RansEncParams {
    const uint8_t *idx;       // [n][h][w][c_y]
    const int16_t *sym;       // [n][h][w][c_y]
    const uint32_t *cf;       // [nb][256]: c[pos] | freq[pos] << 16
    int n_chunks, n_sub, h, w, c_y, rows_per_sub, W, n_buckets;
    uint16_t *tmp_words;      // scratch: [n*n_sub][W/32][tmp_stride] words in emission order
    size_t tmp_stride;
    uint8_t *stage;           // scratch: [n*n_sub][stage_stride] one finished substream each
    size_t stage_stride;
    uint32_t *sizes;          // [n*n_sub] bytes of each substream
    uint8_t *bits_out;        // packed substreams (4-byte aligned), capacity cap
    size_t cap;
    uint32_t *sub_off;        // [n*n_sub + 1] byte offsets into bits_out
    uint32_t *status;
};
cudaError_t launch_rans_encode(const RansEncParams &p, LaunchStream st);
// encode_static.cu: device address, on the CURRENT device, of the file-scope scratch array ufnvc_encode_chunk_dev_static uses
cudaError_t static_scratch_address(void **ptr);
// NEXT-3 (R22): decoded hyper-latent, channels-last int16 [n][pz][c_z] -> the planar [n][c_z][pz] layout of z_dev
cudaError_t launch_z_hwc_to_planar(const int16_t *z_hwc, int16_t *z_planar, int n_chunks, int c_z, int pz, LaunchStream st);

// encoder-side kernels (encode.cu, R24)
cudaError_t launch_enc_patchify(const float *frames, bf16 *out, int n_img, int height, int width, int H8, int W8, LaunchStream st);
cudaError_t launch_hyper_encoder(const float *y, const float *w0, const float *b0, const float *w1, const float *b1, float *a, int16_t *z,
                                 float *zf_tap, int n_img, int h, int w, int hz, int wz, int c_y, int c_h, int c_z, LaunchStream st);
cudaError_t launch_enc_quantise(const float *y, const float *mu, int16_t *sym, long long n, LaunchStream st);
cudaError_t launch_colour(const float *in, float *out, long long plane, long long n_img, bool to_yuv, cudaStream_t st);

// tcgen05 implicit-GEMM conv (conv_tc.cu)
cudaError_t launch_conv_tc(const ConvLayer &L, const ConvProblem &P, const CUtensorMap &tmap_in, int tile_h, int tile_w,
                           bool flat, const EpiParams &E, int num_sms, LaunchStream st);
cudaError_t launch_conv_halo_pair(const ConvLayer &L, const ConvProblem &P, const CUtensorMap &tmap_halo, const EpiParams &E, int num_sms,
                                  LaunchStream st, bool transposed);   // transposed: tmap_halo from tc_make_halo_tmap_transposed
cudaError_t launch_conv_halo(const ConvLayer &L, const ConvProblem &P, const CUtensorMap &tmap_halo, const EpiParams &E, int num_sms,
                             LaunchStream st);
bool tc_make_halo_tmap(CUtensorMap *tm, const bf16 *base, int n_img, int H, int W, int C, std::string &err);
bool tc_make_halo_tmap_transposed(CUtensorMap *tm, const bf16 *base, int n_img, int H, int W, int C, std::string &err);
bool halo_prefers_transposed(int H, int W);   // the 16 x 8 halo tile pads the image to fewer tiles as 8 rows x 16 columns
bool tc_make_weight_tmap(ConvLayer &L, std::string &err, int block_n = 0);   // block_n = 0: widest N tile that divides n_pad
bool tc_make_act_tmap(CUtensorMap *tm, const bf16 *base, int n_img, int H, int W, int C, int tile_h, int tile_w,
                      std::string &err, bool swizzle = true, int pix_stride = 0);   // pix_stride: elements between pixels (0 = C)

bool tc_encode_2d(CUtensorMap *tm, const void *base, unsigned long long dim0, unsigned long long dim1, unsigned box0, unsigned box1,
                  std::string &err);   // 2-D bf16 map, dim0 contiguous, 128B swizzle, zero OOB fill

bool tc_encode_3d(CUtensorMap *tm, const void *base, unsigned long long d0, unsigned long long d1, unsigned long long d2, unsigned b0,
                  unsigned b1, unsigned b2, std::string &err);

// A9, input-stationary (final_tc.cu): 9 taps folded into N, shifted sum of the partial planes in the epilogue
struct FinalMaps {
    CUtensorMap tm_in, tm_w;
    const bf16 *in_base = nullptr;
    bool ok = false;
};
bool final_make_maps(FinalMaps &m, const ConvLayer &L, const bf16 *in_base, int n_img, int H, int W, int out_w, std::string &err);
cudaError_t launch_final_is(const FinalMaps &m, const ConvLayer &L, int n_img, int H, int W, float *out, int out_h, int out_w,
                            int num_sms, LaunchStream st);

// fused trunk MLP (trunk_tc.cu): out = x + W2 GELU(W1 d + b1) + b2 in one kernel, hidden kept on chip
struct TrunkMaps {
    CUtensorMap tm_d, tm_w1, tm_w2, tm_w1h, tm_w2h;   // *h: half tiles for the CTA-pair kernel
    bool ok = false;
};
bool trunk_make_maps(TrunkMaps &m, const bf16 *d_base, long long n_px, const ConvLayer &pw1, const ConvLayer &pw2, std::string &err);
cudaError_t launch_trunk_mlp(const TrunkMaps &m, const ConvLayer &pw1, const ConvLayer &pw2, const bf16 *x, bf16 *out, long long n_px,
                             int num_sms, bool pair, LaunchStream st, uint32_t *tile_done = nullptr, bool quad_clusters = true);
// the CTA-pair trunk kernel adds 1 to tile_done[tile] per drain warp (8) of the CTA that owns the 128-pixel tile: a tile is
// complete (written, and its input rows no longer read) when its counter reaches kTrunkTileSignals
constexpr uint32_t kTrunkTileSignals = 8;
// true if launch_trunk_mlp(..., pair, ...) runs the CTA-pair kernel, the one that counts finished tiles in tile_done
bool trunk_counts_tiles(long long n_px, bool pair);

// rANS symbol search: 128-slot bins, one 32-bit entry each (tables.cu build_search_lut)
constexpr int kLutShift = 7, kLutBuckets = 65536 >> kLutShift;

// ---- host-side entropy tables + encoder fixture (tables.cpp part of api) ---------------------------------------
void build_cdf_tables(int nb, double smin, double smax, std::vector<uint32_t> &cdf32);
void build_search_lut(const std::vector<uint32_t> &cdf32, int nb, std::vector<uint32_t> &lut);
long encode_substream(const uint32_t *cdf32, const uint8_t *idx, const int16_t *sym, size_t n, int W, uint8_t *out,
                      size_t cap);

}  // namespace ufnvc
