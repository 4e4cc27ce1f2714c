/*
 * ufnvc oracle -- TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow CPU restatement of the chunk-decode path of "Ultra-Fast Neural Video
 * Compression" (DCVC-UF, /root/reference/PAPER.md) as fixed by SURVEY.md section 8(c),
 * steps O1..O9.  It shares no code with the CUDA path (paper_2606_04410_b200/csrc) and
 * is imported only by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs.  REAL is double unless -DREAL=float (the "plain fp32" variant
 * BASELINE.json names; the fp32-vs-fp64 pin bounds its own rounding error).
 *
 * All tensors here are planar [C][H][W] per frame, the layout the definitions are written
 * in.  Loops are the definitions themselves: no blocking, no fusion.  OpenMP only splits
 * the outermost independent index.
 *
 * Parity pins (tests/test_oracle_pins.py): CDF closed-form values and invariants,
 * brute-force 7-deep conv in numpy, delta/constant kernels, pixel-shuffle bijection,
 * rANS round trip + end state + size-vs-entropy bound + one-symbol closed form, GELU
 * identities, bucket level values.  Fidelity to the paper's TRAINED codec: parity
 * unpinned (no weights, no data, no worked numerical example in PAPER.md).
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifndef REAL
#define REAL double
#endif

int orc_real_bytes(void) { return (int)sizeof(REAL); }

/* O1/O8: stride-1 cross-correlation, zero padding (k-1)/2, bias.
 * out[o,y,x] = b[o] + sum_{c,dy,dx} w[o,c,dy,dx] * in[c, y+dy-p, x+dx-p],  k in {1,3}. */
void orc_conv2d(const REAL *in, int C_in, int H, int W, const REAL *wt, const REAL *b,
                int C_out, int k, REAL *out)
{
    const int p = (k - 1) / 2;
#pragma omp parallel for schedule(dynamic, 1)
    for (int o = 0; o < C_out; ++o) {
        REAL *dst = out + (size_t)o * H * W;
        for (size_t i = 0; i < (size_t)H * W; ++i) dst[i] = b ? b[o] : (REAL)0;
        for (int c = 0; c < C_in; ++c) {
            const REAL *src = in + (size_t)c * H * W;
            for (int dy = 0; dy < k; ++dy)
                for (int dx = 0; dx < k; ++dx) {
                    const REAL wv = wt[(((size_t)o * C_in + c) * k + dy) * k + dx];
                    for (int y = 0; y < H; ++y) {
                        const int yy = y + dy - p;
                        if (yy < 0 || yy >= H) continue;
                        const int x0 = (p - dx) > 0 ? (p - dx) : 0;
                        const int x1 = (W + p - dx) < W ? (W + p - dx) : W;
                        for (int x = x0; x < x1; ++x)
                            dst[(size_t)y * W + x] += wv * src[(size_t)yy * W + (x + dx - p)];
                    }
                }
        }
    }
}

/* O7: depthwise 3x3, zero pad 1, bias: out[c,y,x] = b[c] + sum_{dy,dx} w[c,0,dy,dx] in[c,y+dy-1,x+dx-1]. */
void orc_dwconv3x3(const REAL *in, int C, int H, int W, const REAL *wt, const REAL *b, REAL *out)
{
#pragma omp parallel for schedule(static)
    for (int c = 0; c < C; ++c)
        for (int y = 0; y < H; ++y)
            for (int x = 0; x < W; ++x) {
                REAL acc = b ? b[c] : (REAL)0;
                for (int dy = 0; dy < 3; ++dy)
                    for (int dx = 0; dx < 3; ++dx) {
                        const int yy = y + dy - 1, xx = x + dx - 1;
                        if (yy < 0 || yy >= H || xx < 0 || xx >= W) continue;
                        acc += wt[(size_t)c * 9 + dy * 3 + dx] * in[((size_t)c * H + yy) * W + xx];
                    }
                out[((size_t)c * H + y) * W + x] = acc;
            }
}

/* O2/O8 [R14]: out[c, r*y+i, r*x+j] = in[c*r*r + i*r + j, y, x];  in is [C*r*r][H][W]. */
void orc_pixel_shuffle(const REAL *in, int C, int H, int W, int r, REAL *out)
{
    const int Ho = H * r, Wo = W * r;
#pragma omp parallel for schedule(static)
    for (int c = 0; c < C; ++c)
        for (int i = 0; i < r; ++i)
            for (int j = 0; j < r; ++j) {
                const REAL *src = in + (size_t)(c * r * r + i * r + j) * H * W;
                for (int y = 0; y < H; ++y)
                    for (int x = 0; x < W; ++x)
                        out[((size_t)c * Ho + (size_t)r * y + i) * Wo + (size_t)r * x + j] = src[(size_t)y * W + x];
            }
}

void orc_relu(REAL *a, size_t n)
{
#pragma omp parallel for schedule(static)
    for (size_t i = 0; i < n; ++i) a[i] = a[i] > 0 ? a[i] : (REAL)0;
}

/* O7/O8: GELU(v) = v/2 * (1 + erf(v / sqrt 2)) -- the exact erf form. */
void orc_gelu(REAL *a, size_t n)
{
#pragma omp parallel for schedule(static)
    for (size_t i = 0; i < n; ++i) {
        const double v = (double)a[i];
        a[i] = (REAL)(0.5 * v * (1.0 + erf(v * 0.70710678118654752440)));
    }
}

/* O2 [R4]: u clamped to [ln smin, ln smax]; idx = clamp(floor((nb-1)*(u-ln smin)/ln(smax/smin) + 0.5)).
 * The decision is taken in double on both sides (R12). */
void orc_bucket_index(const REAL *u, size_t n, int nb, double smin, double smax, uint8_t *idx, REAL *u_clamped)
{
    const double lo = log(smin), hi = log(smax);
    for (size_t i = 0; i < n; ++i) {
        double v = (double)u[i];
        v = v < lo ? lo : (v > hi ? hi : v);
        if (u_clamped) u_clamped[i] = (REAL)v;
        double t = floor((double)(nb - 1) * (v - lo) / (hi - lo) + 0.5);
        int k = (int)t;
        idx[i] = (uint8_t)(k < 0 ? 0 : (k > nb - 1 ? nb - 1 : k));
    }
}

/* O3 [R7,R8]: 255-symbol alphabet s in [-127,127], position p = s+127.
 * sigma_k = smin*(smax/smin)^(k/(nb-1));  F_k(0)=0, F_k(255)=1,
 * F_k(p) = 1/2 erfc(-(p-127.5)/(sigma_k sqrt 2)) for 1<=p<=254;
 * c_k[p] = p + floor((2^16-255) F_k(p) + 1/2), p = 0..255 (c_k[255] = 2^16).  cdf is [nb][256] u32. */
void orc_build_cdf(int nb, double smin, double smax, uint32_t *cdf)
{
    for (int k = 0; k < nb; ++k) {
        const double sigma = smin * pow(smax / smin, nb > 1 ? (double)k / (double)(nb - 1) : 0.0);
        for (int p = 0; p <= 255; ++p) {
            double F;
            if (p == 0) F = 0.0;
            else if (p == 255) F = 1.0;
            else F = 0.5 * erfc(-((double)p - 127.5) / (sigma * 1.41421356237309504880));
            cdf[(size_t)k * 256 + p] = (uint32_t)p + (uint32_t)floor((65536.0 - 255.0) * F + 0.5);
        }
    }
}

/* position p in [0,254] with c[p] <= slot < c[p+1] (linear scan: obviously correct). */
static int find_pos(const uint32_t *c, uint32_t slot)
{
    int p = 0;
    while (p < 254 && c[p + 1] <= slot) ++p;
    return p;
}

/* [R7] inverse-CDF sampling of r from the QUANTISED table with a uniform 16-bit draw. */
void orc_symbols_from_uniform(const uint32_t *cdf, const uint8_t *idx, const uint16_t *u16, size_t n, int16_t *sym)
{
    for (size_t i = 0; i < n; ++i)
        sym[i] = (int16_t)(find_pos(cdf + (size_t)idx[i] * 256, u16[i]) - 127);
}

/*
 * O4 [R6,R9] rANS, 32-bit state in [2^16, 2^32), 16-bit words, 16-bit probabilities.
 * One substream: n symbols in stream order i; W lanes (multiple of 32); lane l = i mod W, step j = i div W;
 * warp-stream g = lanes [32g, 32g+32), each with its own 32 start states and its own run of words.
 * Container: u32 hdr[2G] = {byte offset of warp-stream g, n_words_g}, then for
 * each g: u32 state[32], u16 word[n_words_g], zero-padded to 4 bytes.
 */
long orc_rans_encode_substream(const uint32_t *cdf, const uint8_t *idx, const int16_t *sym, size_t n, int W,
                               uint8_t *out, size_t cap)
{
    const int G = W / 32;
    const size_t steps = (n + (size_t)W - 1) / (size_t)W;
    size_t pos = (size_t)8 * G;
    if (W <= 0 || W % 32 || cap < pos) return -1;
    uint16_t *words = (uint16_t *)malloc((n + 1) * sizeof(uint16_t));   /* <= 1 word per symbol */
    if (!words) return -1;
    for (int g = 0; g < G; ++g) {
        uint64_t x[32];
        size_t nw = 0;
        for (int l = 0; l < 32; ++l) x[l] = 65536u;
        /* encoder = exact mirror of the decoder: steps descending, lanes descending */
        for (size_t jj = steps; jj-- > 0;) {
            for (int l = 31; l >= 0; --l) {
                const size_t i = jj * (size_t)W + (size_t)(32 * g + l);
                if (i >= n) continue;
                const uint32_t *c = cdf + (size_t)idx[i] * 256;
                const int p = (int)sym[i] + 127;
                if (p < 0 || p > 254) { free(words); return -2; }
                const uint64_t f = c[p + 1] - c[p], cs = c[p];
                if (x[l] >= (f << 16)) { words[nw++] = (uint16_t)(x[l] & 0xFFFFu); x[l] >>= 16; }
                x[l] = ((x[l] / f) << 16) + (x[l] % f) + cs;
            }
        }
        while (pos % 4) out[pos++] = 0;
        if (pos + 128 + 2 * nw + 2 > cap) { free(words); return -1; }
        ((uint32_t *)out)[2 * g] = (uint32_t)pos;
        ((uint32_t *)out)[2 * g + 1] = (uint32_t)nw;
        for (int l = 0; l < 32; ++l) { uint32_t v = (uint32_t)x[l]; memcpy(out + pos, &v, 4); pos += 4; }
        for (size_t q = 0; q < nw; ++q) { uint16_t v = words[nw - 1 - q]; memcpy(out + pos, &v, 2); pos += 2; }
    }
    while (pos % 4) out[pos++] = 0;
    free(words);
    return (long)pos;
}

/* returns 0 = OK; 1 = end state != 2^16; 2 = word count mismatch; 3 = header/overrun. */
int orc_rans_decode_substream(const uint32_t *cdf, const uint8_t *idx, size_t n, int W,
                              const uint8_t *in, size_t nbytes, int16_t *sym)
{
    const int G = W / 32;
    const size_t steps = (n + (size_t)W - 1) / (size_t)W;
    int status = 0;
    if (W <= 0 || W % 32 || nbytes < (size_t)8 * G) return 3;
    for (int g = 0; g < G; ++g) {
        uint32_t off, nw;
        memcpy(&off, in + 8 * g, 4);
        memcpy(&nw, in + 8 * g + 4, 4);
        if ((size_t)off + 128 + 2 * (size_t)nw > nbytes) { status = 3; nw = 0; if ((size_t)off + 128 > nbytes) continue; }
        uint32_t x[32];
        for (int l = 0; l < 32; ++l) memcpy(&x[l], in + off + 4 * l, 4);
        const uint8_t *wp = in + off + 128;
        size_t q = 0;
        for (size_t j = 0; j < steps; ++j) {
            for (int l = 0; l < 32; ++l) {
                const size_t i = j * (size_t)W + (size_t)(32 * g + l);
                if (i >= n) continue;
                const uint32_t *c = cdf + (size_t)idx[i] * 256;
                const uint32_t slot = x[l] & 0xFFFFu;
                const int p = find_pos(c, slot);
                sym[i] = (int16_t)(p - 127);
                x[l] = (c[p + 1] - c[p]) * (x[l] >> 16) + slot - c[p];
            }
            for (int l = 0; l < 32; ++l) {       /* ascending lane order */
                const size_t i = j * (size_t)W + (size_t)(32 * g + l);
                if (i >= n) continue;
                if (x[l] < 65536u) {
                    uint16_t wv = 0;
                    if (q < nw) memcpy(&wv, wp + 2 * q, 2);
                    x[l] = (x[l] << 16) | wv;
                    ++q;
                }
            }
        }
        for (int l = 0; l < 32; ++l) if (x[l] != 65536u && !status) status = 1;
        if (q != nw && !status) status = 2;
    }
    return status;
}

/* information content sum_i log2(2^16 / freq_i) in bits -- used by the size-vs-entropy pin. */
double orc_ideal_bits(const uint32_t *cdf, const uint8_t *idx, const int16_t *sym, size_t n)
{
    double bits = 0.0;
    for (size_t i = 0; i < n; ++i) {
        const uint32_t *c = cdf + (size_t)idx[i] * 256;
        const int p = (int)sym[i] + 127;
        bits += 16.0 - log2((double)(c[p + 1] - c[p]));
    }
    return bits;
}

/* threads the OpenMP loops above actually use (reported by bench.py's cpu_baseline) */
#ifdef _OPENMP
#include <omp.h>
int orc_num_threads(void) { return omp_get_max_threads(); }
#else
int orc_num_threads(void) { return 1; }
#endif
