// Epilogue arithmetic and addressing shared by the conv kernels (bias is added by the caller).
#pragma once
#include "ufnvc_internal.h"

namespace ufnvc {

// GELU(v) = v/2 (1 + erf(v/sqrt2)), erf by Abramowitz-Stegun 7.1.26 (|abs err| <= 1.5e-7): one MUFU.RCP, one
// MUFU.EX2 and a degree-5 Horner chain -- far below the bf16 rounding (2^-9 relative) the result is stored with.
__device__ __forceinline__ float gelu_erf(float v)
{
    const float z = fabsf(v) * 0.70710678118654752f;
    const float t = __fdividef(1.0f, fmaf(0.3275911f, z, 1.0f));
    float poly = fmaf(1.061405429f, t, -1.453152027f);
    poly = fmaf(poly, t, 1.421413741f);
    poly = fmaf(poly, t, -0.284496736f);
    poly = fmaf(poly, t, 0.254829592f);
    poly *= t;
    const float e = 1.0f - poly * __expf(-z * z);      // erf(|v|/sqrt2)
    const float erfv = copysignf(e, v);
    return 0.5f * v * (1.0f + erfv);
}

// GELU for the tensor-core epilogues: v/2 (1 + tanh(v (a + b v^2 + c v^4))) with (a, b, c) a least-squares fit of
// atanh(erf(v/sqrt2))/v weighted by the GELU sensitivity (|fit - erf form| <= 3e-5 on the whole line; the classic
// 0.044715 tanh form is off by 4.7e-4), and tanh by MUFU.TANH (relative error 2^-11).  6 FMA-pipe instructions + 1 MUFU
// per element instead of 17 + 2: the epilogue, not the MMAs, bounded the first-pass conv kernels.  v^2 is clamped so
// the fitted polynomial stays in its monotone range (|v| <= 7; tanh is saturated long before).
__device__ __forceinline__ float gelu_fast(float v)
{
    const float s = fminf(v * v, 49.0f);
    float pl = fmaf(-3.58006361e-4f, s, 3.70462883e-2f);
    pl = fmaf(pl, s, 7.97462455e-1f);
    const float u = v * pl;
    float t;
    asm("tanh.approx.f32 %0, %1;" : "=f"(t) : "f"(u));
    const float hv = 0.5f * v;
    return fmaf(hv, t, hv);
}

// Two GELUs at once on the packed-fp32 pipe (sm_100 FADD2 / FMUL2 / FFMA2): (acc0 + b0, acc1 + b1) -> gelu_fast of each.
// 13 issue slots per PAIR (6 packed FMA-pipe ops, 2 FMNMX, 2 MUFU.TANH, + the bf16 pack done by the caller).
__device__ __forceinline__ uint64_t f2_pack(float a, float b)
{
    uint64_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ void f2_unpack(uint64_t v, float &a, float &b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ uint64_t f2_fma(uint64_t a, uint64_t b, uint64_t c)
{
    uint64_t r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ uint64_t f2_mul(uint64_t a, uint64_t b)
{
    uint64_t r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ uint64_t f2_add(uint64_t a, uint64_t b)
{
    uint64_t r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ void gelu_bias2(float acc0, float acc1, float b0, float b1, float &g0, float &g1)
{
    const uint64_t v = f2_add(f2_pack(acc0, acc1), f2_pack(b0, b1));
    float s0, s1;
    f2_unpack(f2_mul(v, v), s0, s1);
    const uint64_t s = f2_pack(fminf(s0, 49.0f), fminf(s1, 49.0f));
    uint64_t pl = f2_fma(f2_pack(-3.58006361e-4f, -3.58006361e-4f), s, f2_pack(3.70462883e-2f, 3.70462883e-2f));
    pl = f2_fma(pl, s, f2_pack(7.97462455e-1f, 7.97462455e-1f));
    float u0, u1, t0, t1;
    f2_unpack(f2_mul(v, pl), u0, u1);
    asm("tanh.approx.f32 %0, %1;" : "=f"(t0) : "f"(u0));
    asm("tanh.approx.f32 %0, %1;" : "=f"(t1) : "f"(u1));
    const uint64_t hv = f2_mul(v, f2_pack(0.5f, 0.5f));
    f2_unpack(f2_fma(hv, f2_pack(t0, t1), hv), g0, g1);
}

__device__ __forceinline__ float apply_act(float v, int act) { return act == ACT_GELU ? gelu_erf(v) : v; }

// Destination element offset of packed output column n of input pixel (img, y, x); EPI_NHWC / EPI_PS2 only.
// 256-bit global store (sm_100: STG.E.256): one thread writes a whole 32-byte sector, so a row that a thread owns never
// reaches L2 as half-sector partial writes (which cost a read-modify-write each).  p must be 32-byte aligned.
__device__ __forceinline__ void st_global_256(void *p, const float *f)
{
    asm volatile("st.global.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "f"(f[0]), "f"(f[1]), "f"(f[2]), "f"(f[3]), "f"(f[4]),
                 "f"(f[5]), "f"(f[6]), "f"(f[7]) : "memory");
}
__device__ __forceinline__ void st_global_256(void *p, const uint32_t *u)
{
    asm volatile("st.global.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "r"(u[0]), "r"(u[1]), "r"(u[2]), "r"(u[3]), "r"(u[4]),
                 "r"(u[5]), "r"(u[6]), "r"(u[7]) : "memory");
}

__device__ __forceinline__ long long epi_offset(const EpiParams &E, int img, int y, int x, int H, int W, int n)
{
    if (E.mode == EPI_NHWC) {
        if (E.unps2)
            return (long long)img * E.img_stride + (((long long)(y >> 1) * (W >> 1) + (x >> 1)) * 4 + ((y & 1) * 2 + (x & 1))) * E.n_split + n;
        const int grp = n / E.n_split, c = n - grp * E.n_split;
        return (long long)img * E.img_stride + (long long)grp * E.split_stride + ((long long)y * W + x) * (E.pix_stride ? E.pix_stride : E.n_split) + c;
    }
    const int ij = n / E.c_o, c = n - ij * E.c_o;
    const int oy = 2 * y + (ij >> 1), ox = 2 * x + (ij & 1);
    return (long long)img * E.img_stride + ((long long)oy * (2 * W) + ox) * E.c_o + c;
}

// EPI_FINAL: clamp, crop, planar fp32 (A9 / O9).
__device__ __forceinline__ void epi_store_final(const EpiParams &E, int img, int y, int x, int n, float v)
{
    const int ij = n / E.c_o, c = n - ij * E.c_o;
    const int oy = 2 * y + (ij >> 1), ox = 2 * x + (ij & 1);
    if (oy >= E.out_h || ox >= E.out_w) return;
    v = fminf(fmaxf(v, 0.0f), 1.0f);
    reinterpret_cast<float *>(E.out)[(long long)img * E.img_stride + ((long long)c * E.out_h + oy) * E.out_w + ox] = v;
}

}  // namespace ufnvc
