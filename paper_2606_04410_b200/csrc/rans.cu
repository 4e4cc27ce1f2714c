// A3 + A4: parallel rANS decode of independent substreams + dequantisation.
// "we can perform arithmetic decoding for all partitions in one consolidated step";
// "r_i is recovered using only sigma_i, and the final latent is reconstructed as y_i = r_i + mu_i".
//
// One thread block per substream, one warp per warp-stream (32 interleaved 32-bit rANS states, 16-bit words,
// 16-bit probabilities).  Per step every lane decodes one symbol; lanes whose state fell below 2^16 pull the next
// words of the warp's word run in ascending lane order -- a ballot + popc prefix (the warp-level scan).  The words
// are kept in a 64-entry register window (two per lane) and fetched with shuffles, so the serial critical path per
// step is: 1 shared-memory LUT read, 1 table read, a few integer ops, 1 ballot, 1 shuffle.  The idx / mu loads of
// step j+1 do not depend on the state and are issued one step ahead.
#include "ufnvc_internal.h"

namespace ufnvc {

__device__ __forceinline__ uint32_t lds_u32(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}
// prefetch loads as volatile asm: the compiler keeps them where they are written (a whole register bank ahead of their use)
// instead of sinking them next to the consumer, where every step would wait for an L2 round trip
__device__ __forceinline__ uint32_t ldg_u8(const uint8_t *p)
{
    uint32_t v;
    asm volatile("ld.global.nc.u8 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ float ldg_f32(const float *p)
{
    float v;
    asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(v) : "l"(p));
    return v;
}

constexpr int kRansWarps = 4;        // warp-streams per block: one per SM sub-partition, so a step's ~90 instructions never queue
                                     // behind another warp's (16 warps per block measured 0.33 us per step, issue-slot bound)

// TAPS: the optional fp32 / int16 outputs exist (parity taps, or the residual the progressive means need).
// STRIDED: y is a channel block of a wider tensor (y_stride != c_y, R23).
// Grid: (substream, group of blockDim.x / 32 warp-streams).
template <bool TAPS, bool STRIDED>
__global__ void __launch_bounds__(32 * kRansWarps) rans_decode_kernel(RansParams p, int nb, int groups_per_sub)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    // tables in shared memory, addressed as 32-bit shared addresses (one LDS per access, no generic-address arithmetic in
    // the serial chain): cf[k][pos] = c[pos] | freq[pos] << 16 (freq <= 65282 fits 16 bits), then the search entries
    const uint32_t s_cf = uint32_t(__cvta_generic_to_shared(smem_raw));
    const uint32_t s_lut = s_cf + uint32_t(nb) * 1024u;
    const uint32_t s_bar = s_lut + uint32_t(nb) * uint32_t(kLutBuckets) * 4u;
    if (threadIdx.x == 0) {
        // the 192 KB of static tables arrive by bulk async copies (one thread, 32 KB pieces) while the predecessor kernel is
        // still running (PDL): nothing here depends on it
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(s_bar) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        const uint32_t cf_bytes = uint32_t(nb) * 1024u, lut_bytes = uint32_t(nb) * uint32_t(kLutBuckets) * 4u;
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(s_bar), "r"(cf_bytes + lut_bytes) : "memory");
        for (uint32_t o = 0; o < cf_bytes; o += 32768u) {
            const uint32_t nbytes = cf_bytes - o < 32768u ? cf_bytes - o : 32768u;
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(s_cf + o),
                         "l"(reinterpret_cast<const unsigned char *>(p.cf) + o), "r"(nbytes), "r"(s_bar) : "memory");
        }
        for (uint32_t o = 0; o < lut_bytes; o += 32768u) {
            const uint32_t nbytes = lut_bytes - o < 32768u ? lut_bytes - o : 32768u;
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(s_lut + o),
                         "l"(reinterpret_cast<const unsigned char *>(p.lut) + o), "r"(nbytes), "r"(s_bar) : "memory");
        }
    }
    // idx, mu, the bit-stream and the status word are only touched after the predecessor grid has completed
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    __syncthreads();                            // the barrier is initialised

    const int sub = blockIdx.x / groups_per_sub;                        // chunk * n_sub + s
    const int chunk = sub / p.n_sub, s = sub % p.n_sub;
    const int g = (blockIdx.x % groups_per_sub) * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    const int G = p.W >> 5;
    const int row0 = s * p.rows_per_sub;
    const int rows = min(p.rows_per_sub, p.h - row0);
    const int n = rows * p.w * p.c_y;                                   // symbols of this substream
    const long long ebase = ((long long)chunk * p.h + row0) * p.w * p.c_y;   // stream order == NHWC order
    const int n_steps = (n + p.W - 1) / p.W;

    // ---- container parsing, every read clamped to the substream ----
    const int so_i = chunk * p.sub_stride + p.sub_first + s;
    const uint32_t so = p.sub_off[so_i], se = p.sub_off[so_i + 1];
    uint32_t st = 0;
    uint32_t sub_bytes = 0;
    if (se < so || (size_t)se > p.bits_bytes || (so & 3)) st |= UFNVC_STREAM_BAD_HEADER; else sub_bytes = se - so;
    const uint8_t *sb = p.bits + so;
    uint32_t ws_off = 0, nw = 0;
    bool ws_ok = false;
    if (sub_bytes >= 8u * G) {
        ws_off = reinterpret_cast<const uint32_t *>(sb)[2 * g];
        nw = reinterpret_cast<const uint32_t *>(sb)[2 * g + 1];
        ws_ok = !(ws_off & 3) && (unsigned long long)ws_off + 128ull + 2ull * nw <= sub_bytes;
    }
    if (!ws_ok) { st |= UFNVC_STREAM_BAD_HEADER; nw = 0; }
    uint32_t x = 1u << 16;
    const uint16_t *words = nullptr;
    if (ws_ok) {
        x = reinterpret_cast<const uint32_t *>(sb + ws_off)[lane];
        words = reinterpret_cast<const uint16_t *>(sb + ws_off + 128);
    }
    // word window: w0/w1/w2 = words[qb + {0,32,64} + lane]; a step consumes <= 32 words and starts with q - qb < 32,
    // so it reads w0/w1 only, and the refill of w2 has a whole window period to land.
    uint32_t qb = 0, q = 0;
    uint32_t w0 = (lane < nw) ? words[lane] : 0u;
    uint32_t w1 = (32u + lane < nw) ? words[32 + lane] : 0u;
    uint32_t w2 = (64u + lane < nw) ? words[64 + lane] : 0u;
    const uint32_t below = (1u << lane) - 1u;

    // idx / mu do not depend on the decoder state: they are fetched kPre steps ahead into two register banks, so the
    // serial chain of a step holds no global-memory latency.  Raw values: nothing consumes them before their step.
    constexpr int kPre = 8;
    const int i0 = g * 32 + lane;
    const uint8_t *idx_p = p.idx + ebase + i0;
    const float *mu_p = p.mu + ebase + i0;
    uint32_t kA[kPre], kB[kPre];
    float mA[kPre], mB[kPre];
    auto fetch = [&](uint32_t (&kk)[kPre], float (&mm)[kPre], int j0) {
#pragma unroll
        for (int t = 0; t < kPre; ++t) {
            const long long o = (long long)(j0 + t) * p.W;
            kk[t] = 0; mm[t] = 0.f;
            if (i0 + o < n) { kk[t] = ldg_u8(idx_p + o); mm[t] = ldg_f32(mu_p + o); }     // (false for every step past the last one, too)
        }
    };
    // running output pointers (element offset of this lane's symbol of the current step)
    long long e_run = ebase + i0;
    // one symbol per lane.  The serial chain: LDS (search entry) -> ~8 integer ops -> LDS (c | freq) -> multiply-add ->
    // compare -> ballot -> popc -> shuffle -> merge.  Everything else (dequantisation, stores) hangs off it.
    auto step = [&](uint32_t k, const float mu, const int j, const bool check) {
        const bool valid = !check || i0 + j * p.W < n;
        // an index past the tables (possible only through idx_override_dev) must not read shared memory out of bounds:
        // clamp and report, like every other malformed input
        if (k >= uint32_t(nb)) { k = uint32_t(nb - 1); st |= UFNVC_STREAM_BAD_HEADER; }
        const uint32_t kofs = k << 10;
        const uint32_t slot = x & 0xFFFFu;
        const uint32_t ent = lds_u32(s_lut + (kofs << 1) + ((slot >> kLutShift) << 2));
        const uint32_t off = slot & ((1u << kLutShift) - 1u);
        const uint32_t lo = ent & 0xFFu, b1 = __byte_perm(ent, 0, 0x4441), b2 = __byte_perm(ent, 0, 0x4442), b3 = ent >> 24;
        uint32_t pos = lo + uint32_t(off >= b1) + uint32_t(off >= b2) + uint32_t(off >= b3);
        if (b1 >= 0xFEu) {                      // > 3 symbols start inside this 128-slot bin (the packed tails)
            if (b1 == 0xFEu) {                  // a run of 1-slot symbols starting at offset b2, b3 of them
                const int t = int(off) - int(b2) + 1;
                pos = lo + uint32_t(min(int(b3), max(t, 0)));
            } else {                            // bisect: largest pos in [lo, lo + b2] with c[pos] <= slot
                uint32_t l = lo, hi = lo + b2;
                while (l < hi) {
                    const uint32_t mid = (l + hi + 1) >> 1;
                    if ((lds_u32(s_cf + kofs + (mid << 2)) & 0xFFFFu) <= slot) l = mid; else hi = mid - 1;
                }
                pos = l;
            }
        }
        const uint32_t cf = lds_u32(s_cf + kofs + (pos << 2));
        uint32_t xn = (cf >> 16) * (x >> 16) + slot - (cf & 0xFFFFu);
        const bool need = valid && xn < (1u << 16);
        const uint32_t m = __ballot_sync(0xFFFFFFFFu, need);
        const uint32_t r = q - qb + __popc(m & below);                   // index into the window, < 64
        const uint32_t wa = __shfl_sync(0xFFFFFFFFu, w0, r & 31);
        const uint32_t wb = __shfl_sync(0xFFFFFFFFu, w1, r & 31);
        if (need) xn = (xn << 16) | (r < 32 ? wa : wb);
        if (valid) x = xn;
        q += __popc(m);
        if (q - qb >= 32) {                     // slide the window (warp-uniform)
            qb += 32;
            w0 = w1; w1 = w2;
            const uint32_t a = qb + 64 + lane;
            w2 = (a < nw) ? words[a] : 0u;
        }
        if (valid) {
            const int sym = int(pos) - 127;
            const float y = float(sym) + mu;                             // O5
            if (!STRIDED) {
                p.yhat[e_run] = __float2bfloat16_rn(y);
            } else {                                                     // y is the first channel block of a wider tensor (R23)
                const long long pix = e_run / p.c_y;
                p.yhat[pix * p.y_stride + (e_run - pix * p.c_y)] = __float2bfloat16_rn(y);
            }
            if (TAPS) {
                if (p.sym_tap) p.sym_tap[e_run] = int16_t(sym);
                if (p.yhat_tap) p.yhat_tap[e_run] = y;
            }
        }
        e_run += p.W;
    };

    const int n_full = n / p.W;                 // steps in which every lane has a symbol
    fetch(kA, mA, 0);
    {                                           // the tables have landed
        uint32_t done = 0;
        while (!done)
            asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0; selp.u32 %0, 1, 0, p; }" : "=r"(done) : "r"(s_bar) : "memory");
    }
    for (int j0 = 0; j0 < n_steps; j0 += 2 * kPre) {
        fetch(kB, mB, j0 + kPre);
        if (j0 + kPre <= n_full) {
#pragma unroll
            for (int t = 0; t < kPre; ++t) step(kA[t], mA[t], j0 + t, false);
        } else {
#pragma unroll
            for (int t = 0; t < kPre; ++t) if (j0 + t < n_steps) step(kA[t], mA[t], j0 + t, true);
        }
        fetch(kA, mA, j0 + 2 * kPre);
        if (j0 + 2 * kPre <= n_full) {
#pragma unroll
            for (int t = 0; t < kPre; ++t) step(kB[t], mB[t], j0 + kPre + t, false);
        } else {
#pragma unroll
            for (int t = 0; t < kPre; ++t) if (j0 + kPre + t < n_steps) step(kB[t], mB[t], j0 + kPre + t, true);
        }
    }
    // end-state invariant (O4): every lane back at 2^16 and every word consumed
    if (__any_sync(0xFFFFFFFFu, x != (1u << 16))) st |= UFNVC_STREAM_BAD_END_STATE;
    if (q != nw) st |= UFNVC_STREAM_BAD_WORD_COUNT;
    st = __reduce_or_sync(0xFFFFFFFFu, st);     // (a clamped index was seen by one lane only)
    if (st && lane == 0) atomicOr(p.status, st);
}

__global__ void z_hwc_to_planar_kernel(const int16_t *__restrict__ in, int16_t *__restrict__ out, int n_chunks, int c_z, int pz)
{
    const long long total = (long long)n_chunks * c_z * pz;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const int p = int(i % pz);                                   // out index: ((n * c_z) + c) * pz + p
        const long long r = i / pz;
        const int c = int(r % c_z);
        const int n = int(r / c_z);
        out[i] = in[((long long)n * pz + p) * c_z + c];
    }
}

cudaError_t launch_z_hwc_to_planar(const int16_t *z_hwc, int16_t *z_planar, int n_chunks, int c_z, int pz, LaunchStream st)
{
    const long long total = (long long)n_chunks * c_z * pz;
    const int blocks = int((total + 255) / 256 < 1184 ? (total + 255) / 256 : 1184);
    z_hwc_to_planar_kernel<<<blocks, 256, 0, st>>>(z_hwc, z_planar, n_chunks, c_z, pz);
    return cudaGetLastError();
}

constexpr size_t kRansSmem = (size_t)64 * (256 * 4 + kLutBuckets * 4) + 16;      // tables + the arrival barrier

cudaError_t configure_rans_kernels()
{
    cudaError_t e = cudaFuncSetAttribute(rans_decode_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRansSmem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(rans_decode_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRansSmem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(rans_decode_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRansSmem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(rans_decode_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRansSmem);
    return e;
}

cudaError_t launch_rans_decode(const RansParams &p, LaunchStream st)
{
    const int nb = p.n_buckets;
    const bool taps = p.sym_tap || p.yhat_tap, strided = p.y_stride != p.c_y;
    const int G = p.W / 32;
    const int wpb = G % kRansWarps == 0 ? kRansWarps : (G % 2 == 0 ? 2 : 1);      // warp-streams per block
    const int groups = G / wpb;
    const unsigned grid = unsigned(p.n_chunks * p.n_sub * groups), block = unsigned(32 * wpb);
    if (taps) return strided ? launch_pdl(rans_decode_kernel<true, true>, grid, block, kRansSmem, st, 1, p, nb, groups)
                             : launch_pdl(rans_decode_kernel<true, false>, grid, block, kRansSmem, st, 1, p, nb, groups);
    return strided ? launch_pdl(rans_decode_kernel<false, true>, grid, block, kRansSmem, st, 1, p, nb, groups)
                   : launch_pdl(rans_decode_kernel<false, false>, grid, block, kRansSmem, st, 1, p, nb, groups);
}

}  // namespace ufnvc
