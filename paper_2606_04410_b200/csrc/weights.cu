// ufnvc_load_weights: parse the blob (include/ufnvc.h), convert / permute / pad, upload.
#include <cmath>
#include <cstring>

#include "handle.h"

namespace ufnvc {

namespace {

struct DirEntry {
    char name[40];
    uint32_t dtype, ndim, shape[4];
    uint64_t offset, nbytes;
};
static_assert(sizeof(DirEntry) == 80, "blob directory entry is 80 bytes");

struct Tensor {
    const uint8_t *data;
    uint32_t dtype, ndim, shape[4];
    size_t count;
    float at(size_t i) const
    {
        if (dtype == 0) { float v; std::memcpy(&v, data + 4 * i, 4); return v; }
        uint16_t b; std::memcpy(&b, data + 2 * i, 2);
        uint32_t u = uint32_t(b) << 16; float v; std::memcpy(&v, &u, 4); return v;
    }
};

uint16_t f32_to_bf16_rne(float f)
{
    uint32_t u; std::memcpy(&u, &f, 4);
    u += 0x7FFFu + ((u >> 16) & 1u);
    return uint16_t(u >> 16);
}

struct Loader {
    ufnvc_handle *h;
    std::map<std::string, Tensor> t;
    std::string err;

    const Tensor *get(const std::string &name, std::initializer_list<uint32_t> shape)
    {
        auto it = t.find(name);
        if (it == t.end()) { err = "missing tensor " + name; return nullptr; }
        const Tensor &x = it->second;
        if (x.ndim != shape.size()) { err = "bad rank for " + name; return nullptr; }
        int d = 0;
        for (uint32_t s : shape) if (x.shape[d++] != s) { err = "bad shape for " + name; return nullptr; }
        return &x;
    }

    template <typename T> T *upload(const std::vector<T> &v)
    {
        T *d = nullptr;
        if (cudaMalloc(&d, v.size() * sizeof(T)) != cudaSuccess) { err = "cudaMalloc failed (weights)"; return nullptr; }
        h->weight_allocs.push_back(d);
        if (cudaMemcpy(d, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice) != cudaSuccess) { err = "cudaMemcpy failed (weights)"; return nullptr; }
        return d;
    }

    // canonical [n][c_in][k][k] (+ bias [n]) for each group -> ConvLayer (bf16 [g][tap][n_pad][c_in], fp32 bias)
    bool conv(ConvLayer &L, const std::vector<std::string> &names, int c_in, int n, int k, bool ps2)
    {
        L.c_in = c_in; L.n = n; L.n_pad = (n + 15) / 16 * 16; L.taps = k * k; L.groups = int(names.size());
        std::vector<uint16_t> w(size_t(L.groups) * L.taps * L.n_pad * c_in, 0);
        std::vector<float> b(size_t(L.groups) * L.n_pad, 0.f);
        const int c_o = n / 4;
        for (int g = 0; g < L.groups; ++g) {
            const Tensor *tw = get(names[g] + ".w", {uint32_t(n), uint32_t(c_in), uint32_t(k), uint32_t(k)});
            const Tensor *tb = get(names[g] + ".b", {uint32_t(n)});
            if (!tw || !tb) return false;
            for (int np = 0; np < n; ++np) {
                const int row = ps2 ? 4 * (np % c_o) + np / c_o : np;       // packed n' = ij*C_o + c  <-  4c + ij
                b[size_t(g) * L.n_pad + np] = tb->at(row);
                for (int tap = 0; tap < L.taps; ++tap)
                    for (int c = 0; c < c_in; ++c)
                        w[((size_t(g) * L.taps + tap) * L.n_pad + np) * c_in + c] =
                            f32_to_bf16_rne(tw->at((size_t(row) * c_in + c) * L.taps + tap));
            }
        }
        L.w = reinterpret_cast<bf16 *>(upload(w));
        L.bias = upload(b);
        L.bias_host = b;
        return L.w && L.bias;
    }

    // Progressive-mean conv k (R21): canonical [c_y][2 c_y][3][3] over [y so far ; mu0].  The kernel feeds y as TWO inputs,
    // y = r + mu with r an integer (exact in bf16) and mu small (bf16 rounding error ~2^-9 |mu|), so the y block of
    // the weights is used twice: device input channels = [r | mu used so far | mu0 | zero pad to a multiple of 64].
    bool mu_net(ConvLayer &L, const std::string &name, int c_y)
    {
        const Tensor *tw = get(name + ".w", {uint32_t(c_y), uint32_t(2 * c_y), 3u, 3u});
        const Tensor *tb = get(name + ".b", {uint32_t(c_y)});
        if (!tw || !tb) return false;
        const int c_in = (3 * c_y + 63) / 64 * 64;
        L.c_in = c_in; L.n = c_y; L.n_pad = (c_y + 15) / 16 * 16; L.taps = 9; L.groups = 1;
        std::vector<uint16_t> w(size_t(9) * L.n_pad * c_in, 0);
        std::vector<float> b(L.n_pad, 0.f);
        for (int o = 0; o < c_y; ++o) {
            b[o] = tb->at(o);
            for (int tap = 0; tap < 9; ++tap)
                for (int c = 0; c < c_y; ++c) {
                    const uint16_t wy = f32_to_bf16_rne(tw->at((size_t(o) * 2 * c_y + c) * 9 + tap));
                    const uint16_t wm = f32_to_bf16_rne(tw->at((size_t(o) * 2 * c_y + c_y + c) * 9 + tap));
                    uint16_t *row = &w[(size_t(tap) * L.n_pad + o) * c_in];
                    row[c] = wy; row[c_y + c] = wy; row[2 * c_y + c] = wm;
                }
        }
        L.w = reinterpret_cast<bf16 *>(upload(w));
        L.bias = upload(b);
        return L.w && L.bias;
    }

    bool hyper(HyperLayer &L, const std::string &name, int c_in, int n)
    {
        const Tensor *tw = get(name + ".w", {uint32_t(n), uint32_t(c_in), 3u, 3u});
        const Tensor *tb = get(name + ".b", {uint32_t(n)});
        if (!tw || !tb) return false;
        L.c_in = c_in; L.n = n;
        std::vector<double> w(size_t(9) * c_in * n), b(n);
        for (int o = 0; o < n; ++o) {
            b[o] = double(tb->at(o));
            for (int c = 0; c < c_in; ++c)
                for (int tap = 0; tap < 9; ++tap) w[(size_t(tap) * c_in + c) * n + o] = double(tw->at((size_t(o) * c_in + c) * 9 + tap));
        }
        L.w = upload(w); L.bias = upload(b);
        return L.w && L.bias;
    }

    // Hybrid head (R12): the last hyper conv on tensor cores with a 2-term bf16 split of its fp64 input
    // (channels [0,c_h) = hi, [c_h,2c_h) = mid, weights duplicated), plus the fp64 weights of the scale half laid out
    // per output row for the exact re-evaluation of elements that land near a bucket edge.
    // packed row n' = (s*16 + 4i+j) * c_y + c2   <-   canonical o = (s*c_y + c2)*16 + 4i+j   (s = 0: mu, 1: ln sigma)
    bool head_hybrid(ConvLayer &L, double *&fix_w, double *&fix_b, float *&wnorm, const std::string &name, int c_h, int c_y)
    {
        const int n = 2 * c_y * 16;
        const Tensor *tw = get(name + ".w", {uint32_t(n), uint32_t(c_h), 3u, 3u});
        const Tensor *tb = get(name + ".b", {uint32_t(n)});
        if (!tw || !tb) return false;
        L.c_in = 2 * c_h; L.n = n; L.n_pad = n; L.taps = 9; L.groups = 1;
        std::vector<uint16_t> w(size_t(9) * n * L.c_in);
        std::vector<float> b(n);
        std::vector<double> fw(size_t(c_y) * 16 * 9 * c_h), fb(size_t(c_y) * 16);
        std::vector<float> wn(n);                                  // |w row|_2, rounded up: input of the head's error bound
        for (int np = 0; np < n; ++np) {
            const int sij = np / c_y, c2 = np % c_y, sft = sij / 16, ij = sij % 16;
            const int o = (sft * c_y + c2) * 16 + ij;
            b[np] = tb->at(o);
            double ss = 0.0;
            for (size_t i = 0; i < size_t(9) * c_h; ++i) { const double v = double(tw->at(size_t(o) * 9 * c_h + i)); ss += v * v; }
            wn[np] = std::nextafter(float(std::sqrt(ss)), INFINITY);
            for (int tap = 0; tap < 9; ++tap)
                for (int c = 0; c < c_h; ++c) {
                    const float v = tw->at((size_t(o) * c_h + c) * 9 + tap);
                    const uint16_t q = f32_to_bf16_rne(v);
                    w[(size_t(tap) * n + np) * L.c_in + c] = q;
                    w[(size_t(tap) * n + np) * L.c_in + c_h + c] = q;
                    if (sft == 1) fw[((size_t(c2) * 16 + ij) * 9 + tap) * c_h + c] = double(v);
                }
            if (sft == 1) fb[size_t(c2) * 16 + ij] = double(tb->at(o));
        }
        L.w = reinterpret_cast<bf16 *>(upload(w));
        L.bias = upload(b);
        fix_w = upload(fw); fix_b = upload(fb); wnorm = upload(wn);
        return L.w && L.bias && fix_w && fix_b && wnorm;
    }

    // R23 fold: canonical [n][T c_t][1][1] -> a conv with T "taps" of c_t channels each (tap t = frame t's feature map)
    bool fold(ConvLayer &L, const std::string &name, int n, int T, int c_t)
    {
        const Tensor *tw = get(name + ".w", {uint32_t(n), uint32_t(T * c_t), 1u, 1u});
        const Tensor *tb = get(name + ".b", {uint32_t(n)});
        if (!tw || !tb) return false;
        L.c_in = c_t; L.n = n; L.n_pad = (n + 15) / 16 * 16; L.taps = T; L.groups = 1;
        std::vector<uint16_t> w(size_t(T) * L.n_pad * c_t, 0);
        std::vector<float> b(L.n_pad, 0.f);
        for (int o = 0; o < n; ++o) {
            b[o] = tb->at(o);
            for (int t = 0; t < T; ++t)
                for (int c = 0; c < c_t; ++c) w[(size_t(t) * L.n_pad + o) * c_t + c] = f32_to_bf16_rne(tw->at(size_t(o) * T * c_t + size_t(t) * c_t + c));
        }
        L.w = reinterpret_cast<bf16 *>(upload(w));
        L.bias = upload(b);
        return L.w && L.bias;
    }

    // R23 prior branch: canonical [c_h][c_ctx][1][1] -> fp64 [c_ctx][c_h] (k-major) + bias
    bool prior(double *&w_p, double *&b_p, const std::string &name, int c_ctx, int c_h)
    {
        const Tensor *tw = get(name + ".w", {uint32_t(c_h), uint32_t(c_ctx), 1u, 1u});
        const Tensor *tb = get(name + ".b", {uint32_t(c_h)});
        if (!tw || !tb) return false;
        std::vector<double> w(size_t(c_ctx) * c_h), b(c_h);
        for (int o = 0; o < c_h; ++o) {
            b[o] = double(tb->at(o));
            for (int k = 0; k < c_ctx; ++k) w[size_t(k) * c_h + o] = double(tw->at(size_t(o) * c_ctx + k));
        }
        w_p = upload(w); b_p = upload(b);
        return w_p && b_p;
    }

    // R24 hyper-encoder: canonical [n][c_in][k][k] -> fp32 [tap][c_in][n] (k-major: a thread per output reads coalesced) + bias
    bool plain(float *&w_d, float *&b_d, const std::string &name, int c_in, int n, int k)
    {
        const Tensor *tw = get(name + ".w", {uint32_t(n), uint32_t(c_in), uint32_t(k), uint32_t(k)});
        const Tensor *tb = get(name + ".b", {uint32_t(n)});
        if (!tw || !tb) return false;
        std::vector<float> w(size_t(k) * k * c_in * n), b(n);
        for (int o = 0; o < n; ++o) {
            b[o] = tb->at(o);
            for (int c = 0; c < c_in; ++c)
                for (int tap = 0; tap < k * k; ++tap) w[(size_t(tap) * c_in + c) * n + o] = tw->at((size_t(o) * c_in + c) * k * k + tap);
        }
        w_d = upload(w); b_d = upload(b);
        return w_d && b_d;
    }

    bool depthwise(float *&dw, float *&db, const std::string &name, int C)
    {
        const Tensor *tw = get(name + ".w", {uint32_t(C), 1u, 3u, 3u});
        const Tensor *tb = get(name + ".b", {uint32_t(C)});
        if (!tw || !tb) return false;
        std::vector<float> w(size_t(9) * C), b(C);
        for (int c = 0; c < C; ++c) {
            b[c] = tb->at(c);
            for (int tap = 0; tap < 9; ++tap) w[size_t(tap) * C + c] = tw->at(size_t(c) * 9 + tap);
        }
        dw = upload(w); db = upload(b);
        return dw && db;
    }
};

}  // namespace

int load_weights_impl(ufnvc_handle *h, const void *blob, size_t bytes)
{
    const uint8_t *p = static_cast<const uint8_t *>(blob);
    if (bytes < 16 || std::memcmp(p, "UFNVCW01", 8) != 0) return fail(h, UFNVC_E_BAD_BLOB, "bad magic");
    uint32_t n_t; std::memcpy(&n_t, p + 8, 4);
    if (n_t > 100000 || 16 + size_t(n_t) * sizeof(DirEntry) > bytes) return fail(h, UFNVC_E_BAD_BLOB, "directory exceeds blob");
    Loader ld; ld.h = h;
    if (!h->weight_allocs.empty()) {                        // a reload replaces the previous weights: nothing may still read them
        cudaDeviceSynchronize();
        for (void *q : h->weight_allocs) cudaFree(q);
        h->weight_allocs.clear();
    }
    for (uint32_t i = 0; i < n_t; ++i) {
        DirEntry e; std::memcpy(&e, p + 16 + size_t(i) * sizeof(DirEntry), sizeof(DirEntry));
        e.name[39] = 0;
        if (e.dtype > 1 || e.ndim < 1 || e.ndim > 4) return fail(h, UFNVC_E_BAD_BLOB, std::string("bad entry ") + e.name);
        size_t cnt = 1; for (uint32_t d = 0; d < e.ndim; ++d) cnt *= e.shape[d];
        const size_t need = cnt * (e.dtype == 0 ? 4 : 2);
        if (e.nbytes != need || e.offset > bytes || need > bytes - e.offset) return fail(h, UFNVC_E_BAD_BLOB, std::string("tensor outside blob: ") + e.name);
        Tensor t{p + e.offset, e.dtype, e.ndim, {e.shape[0], e.shape[1], e.shape[2], e.shape[3]}, cnt};
        ld.t[e.name] = t;
    }
    const ufnvc_config &c = h->cfg;
    bool ok = ld.hyper(h->hyper[0], "hyper.0", c.c_z, c.c_hyper) && ld.hyper(h->hyper[1], "hyper.1", c.c_hyper, c.c_hyper) &&
              ld.hyper(h->hyper[2], "hyper.2", c.c_hyper, 2 * c.c_y * 16);
    if (ok && h->hybrid_head) ok = ld.head_hybrid(h->head_tc, h->head_fix_w, h->head_fix_b, h->head_wnorm, "hyper.2", c.c_hyper, c.c_y);
    ok = ok && ld.conv(h->xframe, {"xframe"}, h->c_cat, c.T * c.c_trunk, 1, false);          // [y ; C_i] with a context (R23)
    for (int k = 1; ok && c.mu_steps == 4 && k <= 3; ++k) ok = ld.mu_net(h->mu_net[k - 1], "mu." + std::to_string(k), c.c_y);
    h->trunk.assign(c.n_trunk_blocks, ufnvc_handle::TrunkBlock());
    const int ce = c.c_trunk * c.trunk_expand;
    for (int k = 0; ok && k < c.n_trunk_blocks; ++k) {
        const std::string b = "trunk." + std::to_string(k);
        ok = ld.depthwise(h->trunk[k].dw_w, h->trunk[k].dw_b, b + ".dw", c.c_trunk) &&
             ld.conv(h->trunk[k].pw1, {b + ".pw1"}, c.c_trunk, ce, 1, false) && ld.conv(h->trunk[k].pw2, {b + ".pw2"}, ce, c.c_trunk, 1, false);
    }
    h->ctx_blocks.assign(c.n_ctx_blocks, ufnvc_handle::TrunkBlock());
    if (ok && h->has_ctx) {
        ok = ld.fold(h->ctx_fold, "ctx.fold", c.c_trunk, c.T, c.c_trunk) && ld.conv(h->ctx_out, {"ctx.out"}, c.c_trunk, c.c_trunk, 1, false) &&
             ld.prior(h->ctx_prior_w, h->ctx_prior_b, "ctx.prior", c.c_trunk, c.c_hyper);
        for (int k = 0; ok && k < c.n_ctx_blocks; ++k) {
            const std::string b = "ctx." + std::to_string(k);
            ok = ld.depthwise(h->ctx_blocks[k].dw_w, h->ctx_blocks[k].dw_b, b + ".dw", c.c_trunk) &&
                 ld.conv(h->ctx_blocks[k].pw1, {b + ".pw1"}, c.c_trunk, ce, 1, false) && ld.conv(h->ctx_blocks[k].pw2, {b + ".pw2"}, ce, c.c_trunk, 1, false);
        }
    }
    h->enc_blocks.assign(c.n_enc_blocks, ufnvc_handle::TrunkBlock());
    if (ok && h->has_enc) {
        ok = ld.conv(h->enc_patch, {"enc.patch"}, 192, c.c_trunk, 1, false) && ld.fold(h->enc_fold, "enc.fold", c.c_trunk, c.T, 4 * c.c_trunk) &&
             ld.conv(h->enc_y, {"enc.y"}, c.c_trunk, c.c_y, 1, false) &&
             ld.plain(h->henc_w0, h->henc_b0, "henc.0", 16 * c.c_y, c.c_hyper, 1) && ld.plain(h->henc_w1, h->henc_b1, "henc.1", c.c_hyper, c.c_z, 3);
        if (ok && h->has_ctx) ok = ld.conv(h->enc_ctx, {"enc.ctx"}, c.c_trunk, c.c_trunk, 1, false);
        for (int k = 0; ok && k < c.n_enc_blocks; ++k) {
            const std::string b = "enc." + std::to_string(k);
            ok = ld.depthwise(h->enc_blocks[k].dw_w, h->enc_blocks[k].dw_b, b + ".dw", c.c_trunk) &&
                 ld.conv(h->enc_blocks[k].pw1, {b + ".pw1"}, c.c_trunk, ce, 1, false) && ld.conv(h->enc_blocks[k].pw2, {b + ".pw2"}, ce, c.c_trunk, 1, false);
        }
    }
    for (int s = 0; ok && s < 4; ++s) {
        std::vector<std::string> names;
        for (int t = 0; t < c.T; ++t) names.push_back("dec." + std::to_string(t) + "." + std::to_string(s));
        ok = ld.conv(h->dec[s], names, c.dec_channels[s], 4 * c.dec_channels[s + 1], 3, true);
    }
    if (!ok) return fail(h, ld.err.find("cuda") == 0 ? UFNVC_E_CUDA : UFNVC_E_BAD_BLOB, ld.err);
    // NEXT-3 (R22), optional: the factorised prior of z -- one ln sigma per channel, bucketed in double by the rule of
    // O2 (hyper.cu), then broadcast to the [n][h_z][w_z][c_z] index map the rANS kernel reads.
    h->z_prior_loaded = false;
    if (ld.t.count("zprior.lnscale")) {
        const Tensor *tz = ld.get("zprior.lnscale", {uint32_t(c.c_z)});
        if (!tz || tz->dtype != 0) return fail(h, UFNVC_E_BAD_BLOB, "zprior.lnscale must be fp32 [c_z]");
        const double lo = std::log(c.scale_min), hi = std::log(c.scale_max);
        h->z_idx_c.resize(c.c_z);
        for (int ch = 0; ch < c.c_z; ++ch) {
            double u = double(tz->at(ch));
            if (!std::isfinite(u)) return fail(h, UFNVC_E_BAD_BLOB, "zprior.lnscale holds a non-finite value");
            u = u < lo ? lo : (u > hi ? hi : u);
            const int k = int(std::floor(double(c.n_buckets - 1) * (u - lo) / (hi - lo) + 0.5));
            h->z_idx_c[ch] = uint8_t(k < 0 ? 0 : (k > c.n_buckets - 1 ? c.n_buckets - 1 : k));
        }
        const size_t cnt = size_t(h->max_chunks) * h->h_z * h->w_z * c.c_z;
        std::vector<uint8_t> full(cnt);
        for (size_t i = 0; i < cnt; ++i) full[i] = h->z_idx_c[i % c.c_z];
        if (cudaMemcpy(h->z_idx, full.data(), cnt, cudaMemcpyHostToDevice) != cudaSuccess) return fail(h, UFNVC_E_CUDA, "cudaMemcpy(z_idx) failed");
        h->z_prior_loaded = true;
    }
    return UFNVC_OK;
}

}  // namespace ufnvc
