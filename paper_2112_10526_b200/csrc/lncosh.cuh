// ln cosh for small arguments (shared by logpsi.cu and pack.cu).
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

}  // namespace nk
