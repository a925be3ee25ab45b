// ln cosh for small arguments and a branch-free fp32 tanh (shared by logpsi.cu, pack.cu and gradient.cu).
#pragma once
#include <cuda_runtime.h>

namespace nk {

// ln cosh t for |t| < 1/2 from its Maclaurin series in u = t^2 (coefficients 2^(2n-1) (2^(2n) - 1) B_2n / (n (2n)!),
// twelve terms: the next one is below 1e-14 at t = 1/2): twelve fp64 FMAs instead of an fp64 exp and log1p.  The five
// configs have |theta| <~ 0.5, so this is the path every element takes there; larger arguments use the stable form.
__device__ __forceinline__ double ln_cosh_small(double t) {
    const double u = t * t;
    double p = -1.6365968284715348e-06;
    p = fma(p, u, 4.405244525877023e-06);
    p = fma(p, u, -1.1956455712177625e-05);
    p = fma(p, u, 3.277930227475478e-05);
    p = fma(p, u, -9.09896491907074e-05);
    p = fma(p, u, 0.0002565805740408915);
    p = fma(p, u, -0.0007386029608251831);
    p = fma(p, u, 0.0021869488536155205);
    p = fma(p, u, -0.006746031746031746);
    p = fma(p, u, 0.022222222222222223);
    p = fma(p, u, -0.08333333333333333);
    p = fma(p, u, 0.5);
    return p * u;
}

// The same series in fp32 (nine terms: the next is below 2e-10 at t = 1/2).  Each term then carries an independent
// rounding error of ~6e-8 of its own size (~0.05), i.e. ~1e-7 over the 2048 terms of config 5, against the 1e-5 bound;
// the sum over hidden units stays in fp64.
__device__ __forceinline__ float ln_cosh_small_f(float t) {
    const float u = t * t;
    float p = 3.277930227475478e-05f;
    p = fmaf(p, u, -9.09896491907074e-05f);
    p = fmaf(p, u, 0.0002565805740408915f);
    p = fmaf(p, u, -0.0007386029608251831f);
    p = fmaf(p, u, 0.0021869488536155205f);
    p = fmaf(p, u, -0.006746031746031746f);
    p = fmaf(p, u, 0.022222222222222223f);
    p = fmaf(p, u, -0.08333333333333333f);
    p = fmaf(p, u, 0.5f);
    return p * u;
}

// ln cosh t for |t| < 1 in fp32: t^2 P(t^2) with P the degree-7 Chebyshev-node least-squares fit of ln cosh(t) / t^2 in
// t^2 on [0, 1] (approximation error 2.2e-10 absolute; fp32 Horner rounding 8e-9 rms, 3.8e-8 at most) — one term fewer
// than the Maclaurin form above on twice its range.  Inf / NaN propagate.
__device__ __forceinline__ float ln_cosh_unit_f(float t) {
    const float u = t * t;
    float p = -2.576627412054222e-05f;
    p = fmaf(p, u, 0.0001767228968674317f);
    p = fmaf(p, u, -0.0006801355048082769f);
    p = fmaf(p, u, 0.002161790616810322f);
    p = fmaf(p, u, -0.00673997588455677f);
    p = fmaf(p, u, 0.02222149446606636f);
    p = fmaf(p, u, -0.08333329856395721f);
    p = fmaf(p, u, 0.5f);
    return p * u;
}

// the two branches of tanh_f32 below, separately (for callers that branch per warp)
__device__ __forceinline__ float tanh_unit_f(float x) {      // |x| < 1
    const float x2 = x * x;
    float p = -0.0003552270936779678f;
    p = fmaf(p, x2, 0.002289985306560993f);
    p = fmaf(p, x2, -0.007930326275527477f);
    p = fmaf(p, x2, 0.021475814282894135f);
    p = fmaf(p, x2, -0.05387599393725395f);
    p = fmaf(p, x2, 0.1333228200674057f);
    p = fmaf(p, x2, -0.33333292603492737f);
    return fmaf(x * x2, p, x);
}
__device__ __forceinline__ float tanh_exp_f(float x) {       // any x; < 2e-7 relative for |x| >= 1
    float E, rc;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(E) : "f"(x * 2.8853900817779268f));
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rc) : "f"(E + 1.f));
    return fmaf(-2.f, rc, 1.f);
}

// tanh in fp32 without branches: |x| < 1 by x + x^3 P(x^2) (P = degree-6 least-squares fit of (tanh x - x) / x^3 in x^2,
// relative error < 1e-7 in fp32), else 1 - 2 / (e^{2x} + 1) with one MUFU.EX2 and one MUFU.RCP (< 2e-7 relative)
__device__ __forceinline__ float tanh_f32(float x) {
    const float x2 = x * x;
    float p = -0.0003552270936779678f;
    p = fmaf(p, x2, 0.002289985306560993f);
    p = fmaf(p, x2, -0.007930326275527477f);
    p = fmaf(p, x2, 0.021475814282894135f);
    p = fmaf(p, x2, -0.05387599393725395f);
    p = fmaf(p, x2, 0.1333228200674057f);
    p = fmaf(p, x2, -0.33333292603492737f);
    const float small = fmaf(x * x2, p, x);
    float E, rc;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(E) : "f"(x * 2.8853900817779268f));
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rc) : "f"(E + 1.f));
    const float big = fmaf(-2.f, rc, 1.f);
    return fabsf(x) < 1.f ? small : big;
}

}  // namespace nk
