/*
 * ufnvc.h -- C ABI of the B200-native chunk-decode library (libufnvc.so).
 *
 * The operation: decode of one chunk of the chunk-based neural video codec of "Ultra-Fast Neural Video
 * Compression" (DCVC-UF).  PAPER.md:79-81 (section 3.1): "the latent representation y_i is parsed from the
 * bit-stream and fed to the chunk decoder, which generates a rich feature F_i ... used by a set of parallel,
 * frame-specific decoders to reconstruct the individual frames {x_i,0 .. x_i,N-1}".
 * (section 3.4): the parameter network predicts the scales of every element in ONE forward pass, "r_i is
 * recovered using only sigma_i, and the final latent is reconstructed as y_i = r_i + mu_i", arithmetic
 * decoding of all partitions is "one consolidated step".  The layer plan is BASELINE.json:configs as read by
 * SURVEY.md section 8(c) O1..O9 and DESIGN.md (readings R0..R18).
 *
 * Conventions
 *   - plain pointers and sizes only; "_dev" = device pointer (cudaMalloc / torch CUDA tensor), "_host" = host.
 *   - every function returns 0 (UFNVC_OK) or a negative ufnvc_status; no exceptions cross the ABI; no globals, no
 *     environment variables: everything that selects a code path is a field of ufnvc_config.
 *   - a handle is used from one host thread and one CUDA stream at a time; it owns weights, CDF tables,
 *     TMA descriptors and a workspace sized at create for max_chunks_per_call.
 *   - ufnvc_chunk_decode only ENQUEUES work on `cuda_stream` (a cudaStream_t passed as void*; NULL = legacy
 *     default stream): it never synchronises, never allocates and never touches the host copy of anything.
 *   - sm_100 only: ufnvc_create fails with UFNVC_E_UNSUPPORTED_DEVICE elsewhere.  There is no CPU fallback.
 */
#ifndef UFNVC_H
#define UFNVC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum ufnvc_status {
    UFNVC_OK = 0,
    UFNVC_E_INVALID_ARG = -1,
    UFNVC_E_BAD_CONFIG = -2,
    UFNVC_E_NO_WEIGHTS = -3,
    UFNVC_E_BAD_BLOB = -4,
    UFNVC_E_UNSUPPORTED_DEVICE = -5,
    UFNVC_E_CUDA = -6,
    UFNVC_E_OOM = -7
} ufnvc_status;

/* device-side bit-stream status bits, OR-ed over all warp-streams of the last call (ufnvc_get_status) */
#define UFNVC_STREAM_BAD_END_STATE 1u /* some lane did not return to 2^16 */
#define UFNVC_STREAM_BAD_WORD_COUNT 2u /* words consumed != words present */
#define UFNVC_STREAM_BAD_HEADER 4u    /* offsets outside the substream; reads were clamped */

typedef struct ufnvc_handle ufnvc_handle; /* opaque */

/* Plain-old-data, versioned by struct_size.  Geometry (R16): frames are padded at
 * the bottom/right to multiples of 32 (the rule that reproduces every BASELINE.json shape: 1080 -> 1088,
 * 2160 -> 2176, 480 -> 480); latent h = H/16, w = W/16; hyper-latent h_z = ceil(h/4), w_z = ceil(w/4) [R2]. */
typedef struct ufnvc_config {
    uint32_t struct_size;        /* = sizeof(ufnvc_config) */
    int32_t T;                   /* frames per chunk (paper's N), >= 1 */
    int32_t height, width;       /* output frame size, e.g. 1080 x 1920 */
    int32_t c_y, c_z;            /* channels of the chunk latent y and of the hyper-latent z */
    int32_t c_hyper;             /* hyper-decoder width (O1) */
    int32_t c_trunk;             /* per-frame feature width after the cross-frame unfold (O6) */
    int32_t n_trunk_blocks;      /* residual DC blocks shared over t (O7), >= 0 */
    int32_t trunk_expand;        /* 1x1 expansion factor inside a DC block (4) */
    int32_t dec_channels[5];     /* frame-decoder channels, dec_channels[0] == c_trunk, dec_channels[4] == 3 */
    int32_t n_buckets;           /* scale buckets (64), log-spaced on [scale_min, scale_max] inclusive [R4] */
    double scale_min, scale_max; /* 0.11, 20 (double: both the tables and the bucket rule depend on them) */
    int32_t rows_per_substream;  /* latent rows per rANS substream (4) [R9] */
    int32_t lanes_per_substream; /* interleaved rANS lanes W per substream, multiple of 32 in [32,512] (default c_y) */
    int32_t max_chunks_per_call; /* independent chunks decoded by one call (1; 4 for config 4) */
    int32_t weight_dtype;        /* dtype of conv weights in the blob: 0 = fp32, 1 = bf16 */
    int32_t mu_steps;            /* 1: the head's mean serves every element (A4); 4: four-step progressive means
                                  * (R21) -- needs c_y % 32 == 0 and the mu.{1,2,3}
                                  * tensors in the blob; three extra conv launches between A4 and A5 */
    uint32_t debug_flags;        /* 0 = the default (fastest) kernels.  OR of UFNVC_DBG_*: each bit swaps one GPU kernel or
                                  * launch mechanism for its slower cross-check variant (never a CPU path).  Per handle;
                                  * the library reads no environment variable and keeps no process-wide state. */
    int32_t n_ctx_blocks;        /* 0: no temporal context (BASELINE.json's layer plans).  > 0: temporal chunk context (PAPER.md:
                                  * 79-81, 125, 356; R23) with that many DC blocks in the cross-chunk context generation
                                  * (11 / 12 / 9 for the paper's HT-S / HT-L / LD): the handle carries the state C_i from call to
                                  * call (ufnvc_reset_context starts a new video).  Needs c_trunk == 256 and the ctx.* tensors. */
    int32_t n_enc_blocks;        /* 0: decoder only.  > 0: the handle also carries the chunk ENCODER (DESIGN.md
                                  * R24) with that many DC blocks (6 / 7 / 3 for the paper's HT-S / HT-L / LD) and ufnvc_chunk_encode
                                  * works.  Needs c_trunk == 256, mu_steps == 1 and the enc.* / henc.* tensors. */
} ufnvc_config;

/* ufnvc_config.debug_flags: A/B and cross-check switches (tests/test_gpu_parity.py runs every one against the oracle) */
#define UFNVC_DBG_FORCE_GENERIC 0x01u   /* every dense conv on the CUDA-core kernel (no tcgen05), all-fp64 hyper head, unfused trunk */
#define UFNVC_DBG_NO_PDL 0x02u          /* plain stream order instead of programmatic dependent launch */
#define UFNVC_DBG_NO_TAIL_FILL 0x04u    /* trunk: whole-grid waits and static tile striding instead of per-tile counters */
#define UFNVC_DBG_FP64_HEAD 0x08u       /* hyper head (A1 layer 3 + A2) entirely on the FP64 pipe instead of tensor cores + fix-up */
#define UFNVC_DBG_NO_CTA_PAIRS 0x10u    /* single-CTA tcgen05 kernels (cta_group::1) for A7 and A8 instead of CTA pairs */
#define UFNVC_DBG_UNFUSED_TRUNK 0x20u   /* A7 as two 1x1 conv launches with the hidden tensor in HBM */
#define UFNVC_DBG_GENERIC_FINAL 0x40u   /* A9 on the output-stationary halo conv kernel instead of the input-stationary one */
#define UFNVC_DBG_PLAIN_DEPTHWISE 0x80u /* A6 on the register-only kernel (no TMA staging, no tile counters) */
#define UFNVC_DBG_NO_TRANSPOSED_TILES 0x100u /* A8 / head: 16 x 8 pixel tiles only (never the 8 x 16 transposed tile map) */
#define UFNVC_DBG_NO_QUAD_CLUSTERS 0x200u /* A7: every cluster one CTA pair (no weight multicast between two pairs) */

/* Optional device buffers that receive intermediates of ufnvc_chunk_decode_ex (parity/debug; any may be NULL).
 * Layouts are the library's own: channels-last. */
typedef struct ufnvc_taps {
    uint32_t struct_size;
    float *mu;          /* [n][h][w][c_y]  mean (O2); with mu_steps == 4 the mean each element used (R21) */
    float *lnscale;     /* [n][h][w][c_y]  clamped ln sigma (O2) */
    uint8_t *idx;       /* [n][h][w][c_y]  bucket index actually used for decoding */
    int16_t *sym;       /* [n][h][w][c_y]  decoded residual r (O4) */
    float *yhat;        /* [n][h][w][c_y]  r + mu before bf16 rounding (O5) */
    uint16_t *f0;       /* bf16 [n][T][h][w][c_trunk]            after the cross-frame unfold (O6) */
    uint16_t *trunk;    /* bf16 [n][T][h][w][c_trunk]            after the trunk (O7) */
    uint16_t *stage[3]; /* bf16 [n][T][2^s h][2^s w][dec_channels[s]], s = 1..3, after decoder stage s (O8) */
} ufnvc_taps;

/* Validate cfg, check the device (cuda:current), allocate tables + workspace.  *out is set on success only. */
int ufnvc_create(const ufnvc_config *cfg, ufnvc_handle **out);

/* Waits for the device, frees everything the handle owns.  The handle must not be used afterwards. */
int ufnvc_destroy(ufnvc_handle *h);

/* Parse, copy and repack the weights blob (host pointer; not retained).  Blob format (little-endian):
 *   char magic[8] = "UFNVCW01"; uint32 n_tensors; uint32 reserved;
 *   n_tensors x { char name[40]; uint32 dtype (0 fp32, 1 bf16); uint32 ndim; uint32 shape[4];
 *                 uint64 offset (from blob start, 16-byte aligned); uint64 nbytes };
 *   data.
 * Tensors (canonical [C_out][C_in][kh][kw], biases fp32 [C_out]): hyper.{0,1,2}.{w,b}, xframe.{w,b},
 * trunk.{k}.{dw,pw1,pw2}.{w,b}, dec.{t}.{s}.{w,b} (t < T, s < 4); with n_ctx_blocks > 0 xframe.w is
 * [T c_trunk][c_y + c_trunk][1][1] (input = [y ; C_i]) and ctx.fold.{w,b} [c_trunk][T c_trunk][1][1],
 * ctx.{k}.{dw,pw1,pw2}.{w,b} (k < n_ctx_blocks, shapes of a trunk block), ctx.out.{w,b} [c_trunk][c_trunk][1][1],
 * ctx.prior.{w,b} [c_hyper][c_trunk][1][1] are required (R23); with n_enc_blocks > 0 enc.patch.{w,b} [c_trunk][192][1][1],
 * enc.fold.{w,b} [c_trunk][T 4 c_trunk][1][1], enc.{k}.{dw,pw1,pw2}.{w,b} (k < n_enc_blocks), enc.y.{w,b} [c_y][c_trunk][1][1],
 * henc.0.{w,b} [c_hyper][16 c_y][1][1], henc.1.{w,b} [c_z][c_hyper][3][3] and, with a context, enc.ctx.{w,b}
 * [c_trunk][c_trunk][1][1] (R24); with mu_steps == 4 mu.{1,2,3}.{w,b}
 * ([c_y][2 c_y][3][3]: input channels [0, c_y) = y decoded so far, [c_y, 2 c_y) = the head's mean); optional
 * zprior.lnscale (fp32 [c_z], see the bytes-only entry points).
 * Missing / mis-shaped tensor: UFNVC_E_BAD_BLOB. */
int ufnvc_load_weights(ufnvc_handle *h, const void *blob_host, size_t bytes);

/* The hot path, one call, everything enqueued on cuda_stream:
 *   z_dev        int16 [n_chunks][c_z][h_z][w_z]                    hyper-latent (already entropy-decoded, R0)
 *   bits_dev     the rANS bit-stream of r for all chunks, 4-byte aligned
 *   sub_off_dev  uint32 [n_chunks * n_sub + 1] byte offsets of the substreams inside bits_dev, multiples of 4
 *   frames_dev   float [n_chunks][T][3][height][width], values in [0,1]     (output, caller-owned)
 * Bit-stream corruption never faults: reads are clamped and a status word is set (ufnvc_get_status). */
int ufnvc_chunk_decode(ufnvc_handle *h, int n_chunks, const int16_t *z_dev, const uint8_t *bits_dev,
                       size_t bits_bytes, const uint32_t *sub_off_dev, float *frames_dev, void *cuda_stream);

/* ---- bytes-only entry points (R22).  The hyper-latent z has a factorised prior: a
 * zero-mean Gaussian per channel with ln sigma = zprior.lnscale[c] (fp32 [c_z], optional blob tensor), bucketed by the
 * rule of O2 onto the SAME tables as y; it is rANS-coded like y: n_sub_z = ceil(h_z / rows_per_substream) substreams
 * of rows_per_substream rows, stream order (row, col, channel), lanes_per_substream lanes.
 * Without zprior.lnscale in the blob these calls return UFNVC_E_NO_WEIGHTS. ---- */

/* z only: sub_off_dev uint32 [n_chunks * n_sub_z + 1]; z_dev int16 [n_chunks][c_z][h_z][w_z] (output). */
int ufnvc_decode_z(ufnvc_handle *h, int n_chunks, const uint8_t *bits_dev, size_t bits_bytes, const uint32_t *sub_off_dev,
                   int16_t *z_dev, void *cuda_stream);

/* One call from bytes to frames: per chunk the container holds the n_sub_z substreams of z, then the n_sub substreams
 * of r; sub_off_dev uint32 [n_chunks * (n_sub_z + n_sub) + 1].  Two more launches than ufnvc_chunk_decode (the z rANS
 * decode and a layout change); the status word ORs both decodes. */
int ufnvc_chunk_decode_bytes(ufnvc_handle *h, int n_chunks, const uint8_t *bits_dev, size_t bits_bytes,
                             const uint32_t *sub_off_dev, float *frames_dev, void *cuda_stream);

/* ---- temporal chunk context (SURVEY.md 8f NEXT-2a, R23; only with n_ctx_blocks > 0, else UFNVC_E_BAD_CONFIG).
 * the chunk decoder's feature F_i "is also propagated to the next chunk to form the next temporal context";
 * the chunk decoder and the prior are conditioned on C_i.  State per chunk slot of a call (slot k of
 * successive calls = successive chunks of video k): C_i, a bf16 tensor [c_trunk] per latent pixel.  ufnvc_chunk_decode
 * (and _ex / _bytes / _profiled with frames) decodes under the current state and replaces it by C_{i+1}; a call that stops
 * after the entropy stage (frames_dev NULL) and ufnvc_entropy_params read the state and leave it alone.  A fresh handle
 * holds the zero context. ---- */

/* C = 0 for the first n_chunks slots (start of a new video).  Asynchronous on cuda_stream. */
int ufnvc_reset_context(ufnvc_handle *h, int n_chunks, void *cuda_stream);
/* Copy the state out / in: ctx_dev bf16 [n_chunks][h][w][c_trunk] (parity hooks: teacher-forced context). */
int ufnvc_get_context(ufnvc_handle *h, int n_chunks, uint16_t *ctx_dev, void *cuda_stream);
int ufnvc_set_context(ufnvc_handle *h, int n_chunks, const uint16_t *ctx_dev, void *cuda_stream);

/* Same, with parity hooks: idx_override_dev / mu_override_dev ([n][h][w][c_y], may be NULL) replace the
 * hyper-decoder's indices / means ("teacher forcing", R12; the entropy-only mode of DESIGN.md);
 * taps (may be NULL) receives intermediates.  frames_dev may be NULL to stop after the entropy stage. */
int ufnvc_chunk_decode_ex(ufnvc_handle *h, int n_chunks, const int16_t *z_dev, const uint8_t *bits_dev,
                          size_t bits_bytes, const uint32_t *sub_off_dev, float *frames_dev, void *cuda_stream,
                          const uint8_t *idx_override_dev, const float *mu_override_dev, const ufnvc_taps *taps);

/* A1 + A2 only: mu, clamped ln sigma, bucket index, each [n][h][w][c_y] on the device (any may be NULL). */
int ufnvc_entropy_params(ufnvc_handle *h, int n_chunks, const int16_t *z_dev, float *mu_dev, float *lnscale_dev,
                         uint8_t *idx_dev, void *cuda_stream);

/* Synchronises cuda_stream-independent: reads the device status word of the last decode (after the caller
 * synchronised the stream).  *device_status = 0 or an OR of UFNVC_STREAM_* bits. */
int ufnvc_get_status(ufnvc_handle *h, uint32_t *device_status);

/* Human-readable text of the last failing call on this handle (never NULL; NULL handle -> static text). */
const char *ufnvc_last_error(const ufnvc_handle *h);

/* Number of this library's kernels one ufnvc_chunk_decode call enqueues (memsets and copies not counted): the count
 * recorded by the last decode on this handle, else the default path's. For bench accounting. */
int ufnvc_launches_per_call(const ufnvc_handle *h, int n_chunks);

/* Per-stage device time of the LAST ufnvc_chunk_decode_profiled call, in microseconds.
 * ufnvc_chunk_decode_profiled = ufnvc_chunk_decode with a cudaEvent after each stage A1+A2, A3+A4, A5, A6+A7
 * (all trunk blocks), A8 (stages 1-3), A9, context generation; it synchronises the stream at the end.  us_out_host[8]: the
 * six stages, then [6] = A6 alone (sum of the depthwise launches, serialised by their own events) when detail != 0 (two
 * more events per trunk block, which cost a few microseconds of launch gaps), else 0; [7] = context generation (R23; 0
 * without a temporal context). */
int ufnvc_chunk_decode_profiled(ufnvc_handle *h, int n_chunks, const int16_t *z_dev, const uint8_t *bits_dev,
                                size_t bits_bytes, const uint32_t *sub_off_dev, float *frames_dev,
                                void *cuda_stream, int detail, float *us_out_host);

/* Debug counters of the last decode / entropy_params call (synchronises the device).  which = 0: number of latent
 * elements whose scale bucket was re-decided in fp64 by the hybrid head (R12); 0 when the head runs all-fp64. */
int ufnvc_debug_counter(ufnvc_handle *h, int which, uint64_t *value_host);

/* ---- encoder-side fixtures (HOST code, not on the timed path): what a sender would run so that bench.py can
 * build a valid bit-stream without the oracle.  The real codec's encoder runs the decoder's prior net
 * (PAPER.md:125), hence idx comes from ufnvc_entropy_params. ---- */

/* Quantised CDF tables the library decodes with: cdf_host uint32 [n_buckets][256], c[0] = 0, c[255] = 2^16 (O3). */
int ufnvc_get_cdf(const ufnvc_handle *h, uint32_t *cdf_host);

/* Inverse-CDF draw of r from the quantised tables with one uniform 16-bit number per element [R7]. */
int ufnvc_symbols_from_uniform(const ufnvc_handle *h, const uint8_t *idx_host, const uint16_t *u16_host, size_t n,
                               int16_t *sym_host);

/* rANS-encode one chunk (mirror of O4).  idx_host, sym_host: [h][w][c_y].  Writes the concatenated substreams
 * to bits_host (capacity cap bytes) and n_sub + 1 byte offsets (relative to bits_host) to sub_off_host.
 * Returns the byte count (> 0) or a negative status (UFNVC_E_INVALID_ARG if cap is too small). */
long ufnvc_encode_chunk(const ufnvc_handle *h, const uint8_t *idx_host, const int16_t *sym_host, uint8_t *bits_host,
                        size_t cap, uint32_t *sub_off_host);

/* GPU rANS ENCODE of r (the entropy-coding half of a chunk encoder; "the result r_i
 * is arithmetically encoded using scale sigma_i").  Exact mirror of the decoder and byte-identical to
 * ufnvc_encode_chunk / the oracle's encoder.  idx_dev uint8, sym_dev int16: [n_chunks][h][w][c_y] on the device;
 * bits_dev (4-byte aligned, capacity cap bytes) receives the substreams of all chunks back to back and sub_off_dev
 * uint32 [n_chunks * n_sub + 1] their byte offsets -- exactly what ufnvc_chunk_decode takes.  A symbol outside
 * [-127, 127] or an index >= n_buckets sets UFNVC_STREAM_BAD_HEADER in the status word; cap too small sets
 * UFNVC_STREAM_BAD_WORD_COUNT and writes offsets only (sub_off_dev[last] = bytes needed).  Asynchronous on cuda_stream;
 * the first call allocates scratch. */
int ufnvc_encode_chunk_dev(ufnvc_handle *h, int n_chunks, const uint8_t *idx_dev, const int16_t *sym_dev, uint8_t *bits_dev,
                           size_t cap, uint32_t *sub_off_dev, void *cuda_stream);

/* The same GPU rANS encode (same arguments, same kernels, byte-identical output) for callers that may not allocate device
 * memory: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The call allocates NOTHING
 * (no cudaMalloc / cudaFree, no allocating library routine): its scratch is a file-scope __device__ array of
 * UFNVC_STATIC_SCRATCH_BYTES inside the library, which every GPU that loads the library holds until the process exits.
 * Limit: the call's scratch -- about 4.1 bytes per symbol of the call (4.22 MB for one 1080p chunk of config 3) -- must
 * fit the array; a larger call (two 1080p chunks, one 4K chunk) returns UFNVC_E_INVALID_ARG with the byte counts in
 * ufnvc_last_error and does nothing.  All calls on all handles of a device SHARE the array and it keeps the previous call's
 * contents (the call clears what must start at zero): two calls that overlap on the GPU -- different streams without an
 * ordering between them -- race on it; serialise them.  Errors and status bits otherwise as for ufnvc_encode_chunk_dev. */
#define UFNVC_STATIC_SCRATCH_BYTES (8u << 20)
int ufnvc_encode_chunk_dev_static(ufnvc_handle *h, int n_chunks, const uint8_t *idx_dev, const int16_t *sym_dev, uint8_t *bits_dev,
                                  size_t cap, uint32_t *sub_off_dev, void *cuda_stream);

/* ---- chunk ENCODE (R24; only with n_enc_blocks > 0, else UFNVC_E_BAD_CONFIG).  PAPER.md:79:
 * the chunk is patch-embedded to 1/8 resolution, conditioned on C_i and distilled by the chunk encoder into one latent y;
 * r = round(y - mu) is coded with sigma, mu and sigma coming from the DECODER's prior net run on the
 * hyper-latent.  One call, everything on cuda_stream:
 *   frames_dev   float [n_chunks][T][3][height][width] in [0,1]                       (input)
 *   bits_dev     the rANS bit-stream ufnvc_chunk_decode takes, capacity cap bytes     (output, 4-byte aligned)
 *   sub_off_dev  uint32 [n_chunks * n_sub + 1]                                        (output)
 *   z_dev        int16 [n_chunks][c_z][h_z][w_z], the hyper-latent                    (output; what ufnvc_chunk_decode takes)
 *   taps         optional intermediates for parity (any pointer may be NULL)
 * Status bits as for ufnvc_encode_chunk_dev.  With a temporal context the call reads the handle's state C_i and leaves it alone:
 * decoding the produced bytes (as an encoder does to stay in step with its decoder) advances it. */
typedef struct ufnvc_enc_taps {
    uint32_t struct_size;
    float *y;      /* [n][h][w][c_y]      unquantised latent (E5) */
    float *zf;     /* [n][c_z][h_z][w_z]  hyper-encoder output before rounding (E6) */
    int16_t *sym;  /* [n][h][w][c_y]      r = round(y - mu) */
    float *mu;     /* [n][h][w][c_y]      the prior net's mean for the coded z */
    uint8_t *idx;  /* [n][h][w][c_y]      its scale bucket */
} ufnvc_enc_taps;
int ufnvc_chunk_encode(ufnvc_handle *h, int n_chunks, const float *frames_dev, uint8_t *bits_dev, size_t cap, uint32_t *sub_off_dev,
                       int16_t *z_dev, const ufnvc_enc_taps *taps, void *cuda_stream);

/* Colour interface (PAPER.md:384 Supp. C: "a unified YUV444 colorspace that serves as a universal interface"; BT.709 for the RGB
 * tests): full-range BT.709 on [0,1] floats, planar [n_img][3][height][width] in and out (in_dev == out_dev allowed).
 * to_yuv != 0: RGB -> YUV444, else YUV444 -> RGB.  Not part of ufnvc_chunk_decode / _encode: the codec's tensors are whatever
 * three-plane signal the caller feeds it. */
int ufnvc_convert_colour(const float *in_dev, float *out_dev, int n_img, int height, int width, int to_yuv, void *cuda_stream);

/* Bucket index of every channel's z prior, uint8 [c_z] (R22). */
int ufnvc_get_z_prior_index(const ufnvc_handle *h, uint8_t *idx_host);

/* rANS-encode the hyper-latent of one chunk (mirror of ufnvc_decode_z).  z_host int16 [c_z][h_z][w_z]; writes the
 * substreams to bits_host and n_sub_z + 1 offsets to sub_off_host; returns the byte count or a negative status. */
long ufnvc_encode_z(const ufnvc_handle *h, const int16_t *z_host, uint8_t *bits_host, size_t cap, uint32_t *sub_off_host);

#ifdef __cplusplus
}
#endif
#endif /* UFNVC_H */
