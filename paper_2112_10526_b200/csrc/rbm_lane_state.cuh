// Per-lane RBM state shared by the fused local-energy kernel and the Metropolis sampler kernel: one warp owns one
// sample / chain, lane l holds hidden units {128 v + 4 l + c : v < V, c < 4} of theta_s = KAPPA * theta in registers
// and evaluates its share of psi'/psi for one row D of the bond-difference table (see fused_eloc.cu for the maths).
#pragma once
#include "nk_internal.h"
#include "ptx_helpers.cuh"

namespace nk {

__device__ __forceinline__ float warp_sum_f(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ float warp_prod_f(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v *= __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// A lane multiplies up to 4 V factors (1 + e) in [1, 2] into four running products and then these together: at V = 32
// (M_pad = 4096) that is 2^128 when every theta is 0 — the uniform state.  The wide variants therefore scale each
// running product by 2^-16 at the middle of the lane's share, in the base product and in every row's product alike,
// so the power of two cancels exactly in every ratio.
constexpr float WIDE_RESCALE = 1.52587890625e-05f;          // 2^-16

// ---- per-row inner loops ---------------------------------------------------------------------------------
template <int V>
struct RealState {
    float4 th[V];      // theta_s
    float qinv;        // 1 / prod_{j in lane} (1 + e_j)

    __device__ __forceinline__ void load(const float* __restrict__ row, int lane, int /*M_pad*/) {
        float p0 = 1.f, p1 = 1.f, p2 = 1.f, p3 = 1.f;
#pragma unroll
        for (int v = 0; v < V; ++v) {
            float4 t = *reinterpret_cast<const float4*>(row + (v * 32 + lane) * 4);
            t.x *= KAPPA; t.y *= KAPPA; t.z *= KAPPA; t.w *= KAPPA;
            th[v] = t;
            p0 = fmaf(p0, ex2_approx(-fabsf(t.x)), p0);
            p1 = fmaf(p1, ex2_approx(-fabsf(t.y)), p1);
            p2 = fmaf(p2, ex2_approx(-fabsf(t.z)), p2);
            p3 = fmaf(p3, ex2_approx(-fabsf(t.w)), p3);
            if (V > 16 && v == 15) { p0 *= WIDE_RESCALE; p1 *= WIDE_RESCALE; p2 *= WIDE_RESCALE; p3 *= WIDE_RESCALE; }
        }
        qinv = 1.f / ((p0 * p1) * (p2 * p3));
    }
    // this lane's share for one row: p = prod_{j in lane} (1+e'_j) (not yet divided by the base product),
    // acc = sum_j (|x'_j| - |x_j|)
    __device__ __forceinline__ void partial_raw(const float* __restrict__ drow, int lane, float s, float& p,
                                                float& acc) const {
        float p0 = 1.f, p1 = 1.f, p2 = 1.f, p3 = 1.f, acc0 = 0.f, acc1 = 0.f;
#pragma unroll
        for (int v = 0; v < V; ++v) {
            const float4 d = *reinterpret_cast<const float4*>(drow + (v * 32 + lane) * 4);
            const float4 t = th[v];
            const float x0 = fmaf(s, d.x, t.x), x1 = fmaf(s, d.y, t.y);
            const float x2 = fmaf(s, d.z, t.z), x3 = fmaf(s, d.w, t.w);
            p0 = fmaf(p0, ex2_approx(-fabsf(x0)), p0);
            p1 = fmaf(p1, ex2_approx(-fabsf(x1)), p1);
            p2 = fmaf(p2, ex2_approx(-fabsf(x2)), p2);
            p3 = fmaf(p3, ex2_approx(-fabsf(x3)), p3);
            acc0 += fabsf(x0) - fabsf(t.x);
            acc1 += fabsf(x1) - fabsf(t.y);
            acc0 += fabsf(x2) - fabsf(t.z);
            acc1 += fabsf(x3) - fabsf(t.w);
            if (V > 16 && v == 15) { p0 *= WIDE_RESCALE; p1 *= WIDE_RESCALE; p2 *= WIDE_RESCALE; p3 *= WIDE_RESCALE; }
        }
        p = (p0 * p1) * (p2 * p3);
        acc = acc0 + acc1;
    }
    // r = prod_{j in lane} (1+e'_j)/(1+e_j)
    __device__ __forceinline__ void partial(const float* __restrict__ drow, int lane, float s, float& r,
                                            float& acc) const {
        float p;
        partial_raw(drow, lane, s, p, acc);
        r = p * qinv;
    }
    // the move was accepted: theta_s <- theta_s + s D (the same fmaf as in partial_raw), base product <- p
    __device__ __forceinline__ void commit(const float* __restrict__ drow, int lane, float s, float p) {
#pragma unroll
        for (int v = 0; v < V; ++v) {
            const float4 d = *reinterpret_cast<const float4*>(drow + (v * 32 + lane) * 4);
            th[v].x = fmaf(s, d.x, th[v].x); th[v].y = fmaf(s, d.y, th[v].y);
            th[v].z = fmaf(s, d.z, th[v].z); th[v].w = fmaf(s, d.w, th[v].w);
        }
        qinv = 1.f / p;
    }
};

// One pending row of a sample: lane partials plus the row's scalars.  Rows are reduced across the warp two at a
// time: after the first exchange (lane ^ 16) the lower half-warp owns row A and the upper half row B, so the
// five butterfly levels cost 10 shuffles per PAIR of rows instead of 10 per row, and the two rows' serial
// reduction latencies overlap.
struct RowPartR {
    float r, acc, ex, coef;     // ex = s * a2 (visible-bias exponent, log2 units)
};
__device__ __forceinline__ float finish_pair(const RowPartR& A, const RowPartR& B, int lane) {
    const bool up = (lane & 16) != 0;
    float rk = up ? B.r : A.r, ak = up ? B.acc : A.acc;
    const float rs = up ? A.r : B.r, as = up ? A.acc : B.acc;
    rk *= __shfl_xor_sync(0xffffffffu, rs, 16);
    ak += __shfl_xor_sync(0xffffffffu, as, 16);
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) {
        rk *= __shfl_xor_sync(0xffffffffu, rk, o);
        ak += __shfl_xor_sync(0xffffffffu, ak, o);
    }
    const float ex = up ? B.ex : A.ex, c = up ? B.coef : A.coef;
    return c * (rk * ex2_approx(fmaf(0.5f, ak, ex)));   // lower half: row A's term, upper half: row B's
}
__device__ __forceinline__ float finish_single(const RowPartR& A) {
    const float r = warp_prod_f(A.r), acc = warp_sum_f(A.acc);
    return A.coef * (r * ex2_approx(fmaf(0.5f, acc, A.ex)));
}

// y - 2 pi rint(y / 2 pi): the fast __sincosf keeps its 2^-21.4 bound only on [-pi, pi] (beyond, its error grows like
// |y| 2^-24), and a trained complex RBM has |Im theta| of order 10 .. 100.  Im theta is wrapped once per sample at load
// and at every accepted move (the per-pair argument is then the wrapped value plus one table entry, |D| <~ 1), the
// exponent's imaginary part once per amplitude.  Two-constant reduction: 2 pi = 6.28125 + 1.9353072e-3 (the first exact
// in 8 bits, so k * 6.28125 is exact for |k| < 2^16).
__device__ __forceinline__ float wrap_pi(float y) {
    const float k = rintf(y * 0.15915494309189535f);
    return fmaf(k, -1.9353071795864769e-3f, fmaf(k, -6.28125f, y));
}
__device__ __forceinline__ float4 wrap_pi4(float4 y) {
    return make_float4(wrap_pi(y.x), wrap_pi(y.y), wrap_pi(y.z), wrap_pi(y.w));
}

template <int V>
struct CplxState {
    float4 tx[V], ty[V];   // Re theta_s (scaled), Im theta (radians)
    float qr, qi;          // 1 / prod_{j in lane} f_j

    static __device__ __forceinline__ void factor(float x, float y, float& p, float& q) {
        const float e = ex2_approx(-fabsf(x));
        float sn, cs;
        __sincosf(y, &sn, &cs);
        p = fmaf(e, cs, cs);                      // (1+e) cos y
        q = fmaf(-e, sn, sn);                     // (1-e) sin y
        q = __int_as_float(__float_as_int(q) ^ (__float_as_int(x) & 0x80000000));   // times sign(x)
    }
    static __device__ __forceinline__ void cmul(float& ar, float& ai, float br, float bi) {
        const float r = fmaf(ar, br, -ai * bi), i = fmaf(ar, bi, ai * br);
        ar = r; ai = i;
    }
    __device__ __forceinline__ void load(const float* __restrict__ row, int lane, int M_pad) {
        float ar = 1.f, ai = 0.f, br = 1.f, bi = 0.f;
#pragma unroll
        for (int v = 0; v < V; ++v) {
            float4 x = *reinterpret_cast<const float4*>(row + (v * 32 + lane) * 4);
            const float4 y = wrap_pi4(*reinterpret_cast<const float4*>(row + M_pad + (v * 32 + lane) * 4));
            x.x *= KAPPA; x.y *= KAPPA; x.z *= KAPPA; x.w *= KAPPA;
            tx[v] = x; ty[v] = y;
            float p, q;
            factor(x.x, y.x, p, q); cmul(ar, ai, p, q);
            factor(x.y, y.y, p, q); cmul(br, bi, p, q);
            factor(x.z, y.z, p, q); cmul(ar, ai, p, q);
            factor(x.w, y.w, p, q); cmul(br, bi, p, q);
            if (V > 8 && v == 7) { ar *= WIDE_RESCALE; ai *= WIDE_RESCALE; br *= WIDE_RESCALE; bi *= WIDE_RESCALE; }
        }
        cmul(ar, ai, br, bi);
        const float inv = 1.f / fmaf(ar, ar, ai * ai);
        qr = ar * inv; qi = -ai * inv;
    }
    // this lane's share: (ar + i ai) = prod_{j in lane} f'_j (not yet divided by the base product),
    // acc = sum_j (|x'_j| - |x_j|)
    __device__ __forceinline__ void partial_raw(const float* __restrict__ drow, int lane, int M_pad, float s,
                                                float& ar, float& ai, float& acc) const {
        float br = 1.f, bi = 0.f;
        ar = 1.f; ai = 0.f; acc = 0.f;
#pragma unroll
        for (int v = 0; v < V; ++v) {
            const float4 dx = *reinterpret_cast<const float4*>(drow + (v * 32 + lane) * 4);
            const float4 dy = *reinterpret_cast<const float4*>(drow + M_pad + (v * 32 + lane) * 4);
            const float4 x = tx[v], y = ty[v];
            float p, q;
            const float x0 = fmaf(s, dx.x, x.x), x1 = fmaf(s, dx.y, x.y);
            const float x2 = fmaf(s, dx.z, x.z), x3 = fmaf(s, dx.w, x.w);
            factor(x0, fmaf(s, dy.x, y.x), p, q); cmul(ar, ai, p, q);
            factor(x1, fmaf(s, dy.y, y.y), p, q); cmul(br, bi, p, q);
            factor(x2, fmaf(s, dy.z, y.z), p, q); cmul(ar, ai, p, q);
            factor(x3, fmaf(s, dy.w, y.w), p, q); cmul(br, bi, p, q);
            acc += (fabsf(x0) - fabsf(x.x)) + (fabsf(x1) - fabsf(x.y));
            acc += (fabsf(x2) - fabsf(x.z)) + (fabsf(x3) - fabsf(x.w));
            if (V > 8 && v == 7) { ar *= WIDE_RESCALE; ai *= WIDE_RESCALE; br *= WIDE_RESCALE; bi *= WIDE_RESCALE; }
        }
        cmul(ar, ai, br, bi);
    }
    __device__ __forceinline__ void partial(const float* __restrict__ drow, int lane, int M_pad, float s, float& ar,
                                            float& ai, float& acc) const {
        partial_raw(drow, lane, M_pad, s, ar, ai, acc);
        cmul(ar, ai, qr, qi);
    }
    // the move was accepted: theta <- theta + s D, base product <- (pr + i pi)
    __device__ __forceinline__ void commit(const float* __restrict__ drow, int lane, int M_pad, float s, float pr,
                                           float pi) {
#pragma unroll
        for (int v = 0; v < V; ++v) {
            const float4 dx = *reinterpret_cast<const float4*>(drow + (v * 32 + lane) * 4);
            const float4 dy = *reinterpret_cast<const float4*>(drow + M_pad + (v * 32 + lane) * 4);
            tx[v].x = fmaf(s, dx.x, tx[v].x); tx[v].y = fmaf(s, dx.y, tx[v].y);
            tx[v].z = fmaf(s, dx.z, tx[v].z); tx[v].w = fmaf(s, dx.w, tx[v].w);
            ty[v].x = fmaf(s, dy.x, ty[v].x); ty[v].y = fmaf(s, dy.y, ty[v].y);
            ty[v].z = fmaf(s, dy.z, ty[v].z); ty[v].w = fmaf(s, dy.w, ty[v].w);
            ty[v] = wrap_pi4(ty[v]);
        }
        const float inv = 1.f / fmaf(pr, pr, pi * pi);
        qr = pr * inv; qi = -pi * inv;
    }
    static __device__ __forceinline__ void cmul_pub(float& ar, float& ai, float br, float bi) { cmul(ar, ai, br, bi); }
};

struct RowPartC {
    float ar, ai, acc, ex_re, ex_im, coef;   // ex_re = s a2_re (log2 units), ex_im = s a2_im (radians)
};
__device__ __forceinline__ void cmul_f(float& ar, float& ai, float br, float bi) {
    const float r = fmaf(ar, br, -ai * bi), i = fmaf(ar, bi, ai * br);
    ar = r; ai = i;
}
__device__ __forceinline__ void finish_c(float ar, float ai, float acc, float ex_re, float ex_im, float c,
                                         float& out_re, float& out_im) {
    const float mag = c * ex2_approx(fmaf(0.5f, acc, ex_re));
    float sn, cs;
    __sincosf(wrap_pi(ex_im), &sn, &cs);
    cmul_f(ar, ai, mag * cs, mag * sn);
    out_re = ar; out_im = ai;
}
__device__ __forceinline__ void finish_pair_c(const RowPartC& A, const RowPartC& B, int lane, float& out_re,
                                              float& out_im) {
    const bool up = (lane & 16) != 0;
    float kr = up ? B.ar : A.ar, ki = up ? B.ai : A.ai, ka = up ? B.acc : A.acc;
    const float sr = up ? A.ar : B.ar, si = up ? A.ai : B.ai, sa = up ? A.acc : B.acc;
    cmul_f(kr, ki, __shfl_xor_sync(0xffffffffu, sr, 16), __shfl_xor_sync(0xffffffffu, si, 16));
    ka += __shfl_xor_sync(0xffffffffu, sa, 16);
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) {
        const float orr = __shfl_xor_sync(0xffffffffu, kr, o), oi = __shfl_xor_sync(0xffffffffu, ki, o);
        cmul_f(kr, ki, orr, oi);
        ka += __shfl_xor_sync(0xffffffffu, ka, o);
    }
    finish_c(kr, ki, ka, up ? B.ex_re : A.ex_re, up ? B.ex_im : A.ex_im, up ? B.coef : A.coef, out_re, out_im);
}
__device__ __forceinline__ void finish_single_c(const RowPartC& A, float& out_re, float& out_im) {
    float ar = A.ar, ai = A.ai, acc = A.acc;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const float orr = __shfl_xor_sync(0xffffffffu, ar, o), oi = __shfl_xor_sync(0xffffffffu, ai, o);
        cmul_f(ar, ai, orr, oi);
        acc += __shfl_xor_sync(0xffffffffu, acc, o);
    }
    finish_c(ar, ai, acc, A.ex_re, A.ex_im, A.coef, out_re, out_im);
}


// ---- product form: psi'/psi = C_row * prod_j (1 + s t_j tau_j), t = tanh(theta) in registers,
// tau = tanh(d) streamed from the table Ttab (pack.cu), C_row = prod_j cosh d_j folded into the row's exponent.
// No MUFU in the pair loop: one FFMA and one FMUL per pair.  s is warp-uniform, so its sign selects one of two loops
// (a negated source operand is free, a multiplication by s would not be).
template <int V>
struct ProdRealState {
    float4 t[V];

    __device__ __forceinline__ void load(const float* __restrict__ row, int lane, int /*M_pad*/) {
#pragma unroll
        for (int v = 0; v < V; ++v) {
            const float4 x = *reinterpret_cast<const float4*>(row + (v * 32 + lane) * 4);
            t[v] = make_float4(tanhf(x.x), tanhf(x.y), tanhf(x.z), tanhf(x.w));
        }
    }
    template <bool NEG>
    __device__ __forceinline__ float partial_s(const float* __restrict__ trow, int lane) const {
        float p0 = 1.f, p1 = 1.f, p2 = 1.f, p3 = 1.f;
#pragma unroll
        for (int v = 0; v < V; ++v) {
            const float4 d = *reinterpret_cast<const float4*>(trow + (v * 32 + lane) * 4);
            const float4 a = t[v];
            p0 *= fmaf(NEG ? -a.x : a.x, d.x, 1.f);
            p1 *= fmaf(NEG ? -a.y : a.y, d.y, 1.f);
            p2 *= fmaf(NEG ? -a.z : a.z, d.z, 1.f);
            p3 *= fmaf(NEG ? -a.w : a.w, d.w, 1.f);
        }
        return (p0 * p1) * (p2 * p3);
    }
    // partial_s of one row and, in the same basic block, the butterfly of the row pair (da, db) that was completed
    // one step earlier: the shuffles of that reduction (a dependent chain of five) issue between this row's loads and
    // the multiplications that wait for them, instead of leaving the warp without loads in flight.  rk: the product
    // of row a on the lower half-warp, of row b on the upper.
    template <bool NEG>
    __device__ __forceinline__ float partial_s_retire(const float* __restrict__ trow, int lane, float da, float db,
                                                      float& rk) const {
        const bool up = (lane & 16) != 0;
        float k = up ? db : da;
        k *= __shfl_xor_sync(0xffffffffu, up ? da : db, 16);
        float p0 = 1.f, p1 = 1.f, p2 = 1.f, p3 = 1.f;
#pragma unroll
        for (int v = 0; v < V; ++v) {
            const float4 d = *reinterpret_cast<const float4*>(trow + (v * 32 + lane) * 4);
            const float4 a = t[v];
            p0 *= fmaf(NEG ? -a.x : a.x, d.x, 1.f);
            p1 *= fmaf(NEG ? -a.y : a.y, d.y, 1.f);
            p2 *= fmaf(NEG ? -a.z : a.z, d.z, 1.f);
            p3 *= fmaf(NEG ? -a.w : a.w, d.w, 1.f);
            if (v == V / 4) k *= __shfl_xor_sync(0xffffffffu, k, 8);
            if (v == V / 2) k *= __shfl_xor_sync(0xffffffffu, k, 4);
            if (v == (3 * V) / 4) k *= __shfl_xor_sync(0xffffffffu, k, 2);
        }
        k *= __shfl_xor_sync(0xffffffffu, k, 1);
        rk = k;
        return (p0 * p1) * (p2 * p3);
    }
    __device__ __forceinline__ void partial(const float* __restrict__ trow, int lane, float s, float& r,
                                            float& acc) const {
        r = (s > 0.f) ? partial_s<false>(trow, lane) : partial_s<true>(trow, lane);
        acc = 0.f;
    }
};

template <int V>
struct ProdCplxState {
    float4 tr[V], ti[V];

    static __device__ __forceinline__ void ctanh(float x, float y, float& re, float& im) {
        // tanh(x + i y) = [sign(x)(1 - e^2) + i 2 e sin 2y] / (1 + e^2 + 2 e cos 2y),  e = exp(-2|x|)
        const float e = expf(-2.f * fabsf(x));
        float sn, cs;
        sincosf(2.f * y, &sn, &cs);
        const float den = 1.f / (1.f + e * e + 2.f * e * cs);
        re = copysignf((1.f - e) * (1.f + e), x) * den;
        im = 2.f * e * sn * den;
    }
    __device__ __forceinline__ void load(const float* __restrict__ row, int lane, int M_pad) {
#pragma unroll
        for (int v = 0; v < V; ++v) {
            const float4 x = *reinterpret_cast<const float4*>(row + (v * 32 + lane) * 4);
            const float4 y = *reinterpret_cast<const float4*>(row + M_pad + (v * 32 + lane) * 4);
            ctanh(x.x, y.x, tr[v].x, ti[v].x); ctanh(x.y, y.y, tr[v].y, ti[v].y);
            ctanh(x.z, y.z, tr[v].z, ti[v].z); ctanh(x.w, y.w, tr[v].w, ti[v].w);
        }
    }
    // (pr + i pi) *= 1 + s (a_r + i a_i)(d_r + i d_i)
    template <bool NEG>
    static __device__ __forceinline__ void step(float& pr, float& pi, float a_r, float a_i, float d_r, float d_i) {
        const float xr = fmaf(NEG ? a_i : -a_i, d_i, fmaf(NEG ? -a_r : a_r, d_r, 1.f));
        const float xi = fmaf(NEG ? -a_i : a_i, d_r, (NEG ? -a_r : a_r) * d_i);
        const float nr = fmaf(pr, xr, -pi * xi), ni = fmaf(pr, xi, pi * xr);
        pr = nr; pi = ni;
    }
    template <bool NEG>
    __device__ __forceinline__ void partial_s(const float* __restrict__ trow, int lane, int M_pad, float& ar,
                                              float& ai) const {
        float br = 1.f, bi = 0.f;
        ar = 1.f; ai = 0.f;
#pragma unroll
        for (int v = 0; v < V; ++v) {
            const float4 dr = *reinterpret_cast<const float4*>(trow + (v * 32 + lane) * 4);
            const float4 di = *reinterpret_cast<const float4*>(trow + M_pad + (v * 32 + lane) * 4);
            step<NEG>(ar, ai, tr[v].x, ti[v].x, dr.x, di.x);
            step<NEG>(br, bi, tr[v].y, ti[v].y, dr.y, di.y);
            step<NEG>(ar, ai, tr[v].z, ti[v].z, dr.z, di.z);
            step<NEG>(br, bi, tr[v].w, ti[v].w, dr.w, di.w);
        }
        const float r = fmaf(ar, br, -ai * bi), i = fmaf(ar, bi, ai * br);
        ar = r; ai = i;
    }
    __device__ __forceinline__ void partial(const float* __restrict__ trow, int lane, int M_pad, float s, float& ar,
                                            float& ai, float& acc) const {
        if (s > 0.f) partial_s<false>(trow, lane, M_pad, ar, ai);
        else partial_s<true>(trow, lane, M_pad, ar, ai);
        acc = 0.f;
    }
};

// product-form row reductions: as finish_pair / finish_pair_c without the acc butterflies (acc = 0)
__device__ __forceinline__ float finish_pair_prod(const RowPartR& A, const RowPartR& B, int lane) {
    const bool up = (lane & 16) != 0;
    float rk = up ? B.r : A.r;
    const float rs = up ? A.r : B.r;
    rk *= __shfl_xor_sync(0xffffffffu, rs, 16);
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) rk *= __shfl_xor_sync(0xffffffffu, rk, o);
    return (up ? B.coef : A.coef) * (rk * ex2_approx(up ? B.ex : A.ex));
}
__device__ __forceinline__ float finish_single_prod(const RowPartR& A) {
    return A.coef * (warp_prod_f(A.r) * ex2_approx(A.ex));
}
__device__ __forceinline__ void finish_pair_prod_c(const RowPartC& A, const RowPartC& B, int lane, float& out_re,
                                                   float& out_im) {
    const bool up = (lane & 16) != 0;
    float kr = up ? B.ar : A.ar, ki = up ? B.ai : A.ai;
    const float sr = up ? A.ar : B.ar, si = up ? A.ai : B.ai;
    cmul_f(kr, ki, __shfl_xor_sync(0xffffffffu, sr, 16), __shfl_xor_sync(0xffffffffu, si, 16));
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) {
        const float orr = __shfl_xor_sync(0xffffffffu, kr, o), oi = __shfl_xor_sync(0xffffffffu, ki, o);
        cmul_f(kr, ki, orr, oi);
    }
    finish_c(kr, ki, 0.f, up ? B.ex_re : A.ex_re, up ? B.ex_im : A.ex_im, up ? B.coef : A.coef, out_re, out_im);
}
__device__ __forceinline__ void finish_single_prod_c(const RowPartC& A, float& out_re, float& out_im) {
    float ar = A.ar, ai = A.ai;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const float orr = __shfl_xor_sync(0xffffffffu, ar, o), oi = __shfl_xor_sync(0xffffffffu, ai, o);
        cmul_f(ar, ai, orr, oi);
    }
    finish_c(ar, ai, 0.f, A.ex_re, A.ex_im, A.coef, out_re, out_im);
}

}  // namespace nk
