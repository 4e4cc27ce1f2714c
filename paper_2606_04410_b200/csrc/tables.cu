// Host-side entropy-model tables and the encoder-side fixture of libufnvc.
//   * quantised discretised-Gaussian CDF tables, one per scale bucket (readings R7/R8)
//   * the search accelerator the rANS decode kernel uses (slot >> 7 -> position, see build_search_lut)
//   * the rANS ENCODER (mirror of O4), used by callers that need a valid bit-stream (bench.py, tests)
// r = round(y - mu) "is arithmetically encoded using scale sigma".
#include <algorithm>
#include <cmath>
#include <cstring>

#include "ufnvc_internal.h"

namespace ufnvc {

// sigma_k = smin (smax/smin)^(k/(nb-1)); alphabet r in [-127,127] at position p = r + 127;
// c_k[p] = p + round_half_up((2^16 - 255) * Phi((p - 127.5)/sigma_k)), tails folded into the end symbols.
void build_cdf_tables(int nb, double smin, double smax, std::vector<uint32_t> &cdf32)
{
    cdf32.assign((size_t)nb * 256, 0u);
    const double ratio = smax / smin;
    for (int k = 0; k < nb; ++k) {
        const double sigma = smin * std::pow(ratio, nb > 1 ? double(k) / double(nb - 1) : 0.0);
        uint32_t *c = &cdf32[(size_t)k * 256];
        c[0] = 0u;
        c[255] = 65536u;
        for (int p = 1; p <= 254; ++p) {
            const double t = (double(p) - 127.5) / (sigma * 1.41421356237309504880);
            const double Phi = 0.5 * std::erfc(-t);
            c[p] = uint32_t(p) + uint32_t(std::floor(65281.0 * Phi + 0.5));
        }
    }
}

// Search accelerator of the decode kernel.  For every table and every bin b of 2^kLutShift = 128 slots, one 32-bit entry:
//   byte 0      lo = the position holding slot 128 b (largest p with c[p] <= 128 b)
//   bytes 1..3  d_i = c[lo + i] - 128 b for the (at most three) further positions that START inside the bin, 0x80 when
//               there is none: the position of slot 128 b + off is  lo + (off >= d_1) + (off >= d_2) + (off >= d_3)
//               -- no second table access and no loop.
//   more than three starts inside the bin (only where the tails' 1-slot symbols are packed: < 0.5 % of the mass):
//     - the starts are CONSECUTIVE slots d, d + 1, .., d + m - 1 (a run of 1-slot symbols, the far tails of every table):
//               byte 1 = 0xFE, byte 2 = d, byte 3 = m:   position = lo + min(m, max(0, off - d + 1))
//     - otherwise byte 1 = 0xFF, byte 2 = m; the kernel then bisects [lo, lo + m].
void build_search_lut(const std::vector<uint32_t> &cdf32, int nb, std::vector<uint32_t> &lut)
{
    lut.assign((size_t)nb * kLutBuckets, 0u);
    for (int k = 0; k < nb; ++k) {
        const uint32_t *c = &cdf32[(size_t)k * 256];
        int p = 0;
        for (int b = 0; b < kLutBuckets; ++b) {
            const uint32_t s0 = uint32_t(b) << kLutShift, s1 = s0 + (1u << kLutShift) - 1u;
            while (p < 254 && c[p + 1] <= s0) ++p;
            const int lo = p;
            int q = p;
            while (q < 254 && c[q + 1] <= s1) ++q;
            const int m = q - lo;
            uint32_t e = uint32_t(lo);
            if (m <= 3) {
                for (int i = 1; i <= 3; ++i) e |= (i <= m ? c[lo + i] - s0 : 0x80u) << (8 * i);
            } else {
                bool run = m <= 255;
                for (int i = 2; run && i <= m; ++i) run = c[lo + i] == c[lo + 1] + uint32_t(i - 1);
                if (run) e |= 0xFEu << 8 | (c[lo + 1] - s0) << 16 | uint32_t(m) << 24;
                else e |= 0xFFu << 8 | uint32_t(m) << 16 | 0x80u << 24;
            }
            lut[(size_t)k * kLutBuckets + b] = e;
        }
    }
}

// One substream: symbols in stream order, W interleaved lanes, G = W/32 warp-streams.
// Container: u32 hdr[2G] = {byte offset, n_words} per warp-stream; then per warp-stream 32 u32 start states
// followed by its 16-bit words in decode order, each warp-stream 4-byte aligned.
long encode_substream(const uint32_t *cdf32, const uint8_t *idx, const int16_t *sym, size_t n, int W, uint8_t *out,
                      size_t cap)
{
    if (W <= 0 || (W & 31)) return UFNVC_E_INVALID_ARG;
    const int G = W / 32;
    size_t pos = size_t(8) * G;
    if (cap < pos) return UFNVC_E_INVALID_ARG;
    std::vector<uint16_t> emitted;
    emitted.reserve(n / G + 64);
    for (int g = 0; g < G; ++g) {
        uint32_t state[32];
        std::fill(state, state + 32, 1u << 16);
        emitted.clear();
        // Walk this warp-stream's symbols in exactly the reverse of the decoder's visiting order.
        const size_t n_steps = (n + W - 1) / W;
        for (size_t step = n_steps; step > 0; --step) {
            const size_t base = (step - 1) * size_t(W) + size_t(32) * g;
            for (int lane = 31; lane >= 0; --lane) {
                const size_t i = base + lane;
                if (i >= n) continue;
                const int p = int(sym[i]) + 127;
                if (p < 0 || p > 254) return UFNVC_E_INVALID_ARG;
                const uint32_t *c = cdf32 + size_t(idx[i]) * 256;
                const uint32_t start = c[p], freq = c[p + 1] - c[p];
                uint32_t x = state[lane];
                if ((x >> 16) >= freq) {   // x >= freq * 2^16: shed 16 bits first
                    emitted.push_back(uint16_t(x));
                    x >>= 16;
                }
                state[lane] = ((x / freq) << 16) + (x % freq) + start;
            }
        }
        while (pos & 3) out[pos++] = 0;
        const size_t need = 128 + 2 * emitted.size();
        if (pos + need + 4 > cap) return UFNVC_E_INVALID_ARG;
        const uint32_t hdr[2] = {uint32_t(pos), uint32_t(emitted.size())};
        std::memcpy(out + 8 * g, hdr, 8);
        std::memcpy(out + pos, state, 128);
        pos += 128;
        for (size_t q = emitted.size(); q > 0; --q) {
            std::memcpy(out + pos, &emitted[q - 1], 2);
            pos += 2;
        }
    }
    while (pos & 3) out[pos++] = 0;
    return long(pos);
}

}  // namespace ufnvc
