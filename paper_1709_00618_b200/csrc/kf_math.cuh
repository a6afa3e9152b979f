// fp32 Kalman-filter arithmetic of S5 (track following with "a simplified Kalman filter"; only Bz is
// respected).  State p = (y, z, sinPhi, dz/ds, q/pt) at a pad-row plane x; covariance as the packed
// lower triangle c00 c10 c11 c20 c21 c22 c30 c31 c32 c33 c40 c41 c42 c43 c44.  Formulas: DESIGN.md "S5".
// Written from the formulas, not from the oracle's code: the oracle works on full 5x5 fp64 matrices with generic
// loops, this file on the 15 packed fp32 entries with the sparse Jacobian multiplied out by hand.
#pragma once
#include "tpc_common.cuh"

namespace tpc {

struct KfState {
    float y, z, s, t, k;
    float c00, c10, c11, c20, c21, c22, c30, c31, c32, c33, c40, c41, c42, c43, c44;
};

// MUFU approximations with flushed denormals: one instruction each (the default rsqrtf / __fdividef wrap the same
// unit in a denormal rescue of three to four more).  Every argument below is a normal number by construction
// (1 - s^2 >= 0.0975, 1 + tg^2 >= 1, c0 + c1 >= 0.6, S >= sigma^2).
__device__ __forceinline__ float rsqrt_ftz(float x) {
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float rcp_ftz(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// asin(a)/a: arc length over chord for half-angle sine a
__device__ __forceinline__ float asin_over(float a) {
    const float a2 = a * a;
    if (a2 < 0.01f)  // |a| < 0.1: series, truncation < 4e-10
        return 1.0f + a2 * (1.0f / 6.0f + a2 * (3.0f / 40.0f + a2 * (15.0f / 336.0f)));
    return asinf(a) / a;
}

// Transport to the plane x + dx along the exact helix for constant Bz.  Returns false (state untouched) when
// |sinPhi| would leave [-max_s, max_s].
__device__ __forceinline__ bool kf_transport(KfState& st, float dx, float cB, float max_s) {
    const float s = st.s, t = st.t;
    const float kap = cB * st.k;
    const float s1 = fmaf(kap, dx, s);
    if (fmaxf(fabsf(s), fabsf(s1)) > max_s) return false;
    const float c0sq = (1.0f - s) * (1.0f + s), c1sq = (1.0f - s1) * (1.0f + s1);
    const float ic0 = rsqrt_ftz(c0sq), ic1 = rsqrt_ftz(c1sq);
    const float c0 = c0sq * ic0, c1 = c1sq * ic1;
    const float tg = (s + s1) * rcp_ftz(c0 + c1);
    const float sec2 = fmaf(tg, tg, 1.0f);
    const float isec = rsqrt_ftz(sec2);  // sec2 >= 1
    const float chord = dx * (sec2 * isec);
    const float hk = 0.5f * kap;
    const float a = hk * chord;  // sine of half the turning angle
    const float a2 = a * a;
    const float tdx = tg * dx;
    // Path length dS = chord * asin(a)/a, and d(dS)/d(kappa) = (dx/c1 - dS)/kappa.  That difference cancels for small
    // kappa*dx, and the entry steers q/pt through the z residuals, so it is evaluated in a cancellation-free form:
    // with m the chord direction (tan m = tg), h = kappa dS / 2 the half turning angle,
    //   dx/c1 - dS = 2 [cos m (sin h - h cos h) + h sin m sin h] / (kappa c1),
    // and sin h - h cos h = h^3/3 (1 - h^2/10 + h^4/280 - h^6/15120 ...).  Dividing by kappa analytically:
    //   ddS = [tg dx dS / 2 + kappa dS^3 / (12 sqrt(sec2)) (1 - h^2/10 + ...)] / c1.
    float dS, ddS;
    if (a2 < 0.01f) {  // |a| < 0.1, every row-to-row step: both series, truncation < 4e-10 (h^2 < 0.0101: h^6 term < 1e-10)
        dS = chord * fmaf(a2, fmaf(a2, fmaf(a2, 15.0f / 336.0f, 3.0f / 40.0f), 1.0f / 6.0f), 1.0f);
        const float hh = hk * dS, h2 = hh * hh;
        const float ser = fmaf(h2, fmaf(h2, 1.0f / 280.0f, -0.1f), 1.0f);
        ddS = fmaf(0.5f * tdx, dS, (kap * dS) * (dS * dS) * ((1.0f / 12.0f) * isec) * ser) * ic1;
    } else {  // long steps (phase 2: back transports, sector changes)
        dS = chord * (asinf(a) / a);
        const float hh = hk * dS, h2 = hh * hh;
        if (h2 < 0.09f) {
            const float ser = 1.0f + h2 * (-0.1f + h2 * (1.0f / 280.0f - h2 * (1.0f / 15120.0f)));
            ddS = (0.5f * tdx * dS + kap * dS * dS * dS * (1.0f / 12.0f) * isec * ser) * ic1;
        } else {
            ddS = (dx * ic1 - dS) / kap;
        }
    }
    // Jacobian entries (identity elsewhere)
    const float hx = 0.5f * dx * sec2;
    const float f24 = cB * dx;
    const float f02 = hx * (ic0 + ic1);
    const float f04 = f24 * hx * ic1;
    const float f12 = t * tdx * (ic0 * ic1);
    const float f13 = dS;
    const float f14 = cB * t * ddS;
    st.y = fmaf(dx, tg, st.y);
    st.z = fmaf(t, dS, st.z);
    st.s = s1;
    // P <- F P F^T, multiplied out for the lower triangle
    const float n40 = st.c40 + f02 * st.c42 + f04 * st.c44;
    const float n41 = st.c41 + f12 * st.c42 + f13 * st.c43 + f14 * st.c44;
    const float n42 = st.c42 + f24 * st.c44;
    const float n30 = st.c30 + f02 * st.c32 + f04 * st.c43;
    const float n31 = st.c31 + f12 * st.c32 + f13 * st.c33 + f14 * st.c43;
    const float n32 = st.c32 + f24 * st.c43;
    const float a00 = st.c00 + f02 * st.c20 + f04 * st.c40;
    const float a02 = st.c20 + f02 * st.c22 + f04 * st.c42;
    const float a10 = st.c10 + f12 * st.c20 + f13 * st.c30 + f14 * st.c40;
    const float a11 = st.c11 + f12 * st.c21 + f13 * st.c31 + f14 * st.c41;
    const float a12 = st.c21 + f12 * st.c22 + f13 * st.c32 + f14 * st.c42;
    const float a20 = st.c20 + f24 * st.c40;
    const float a21 = st.c21 + f24 * st.c41;
    const float a22 = st.c22 + f24 * st.c42;
    st.c00 = a00 + f02 * a02 + f04 * n40;
    st.c10 = a10 + f02 * a12 + f04 * n41;
    st.c11 = a11 + f12 * a12 + f13 * n31 + f14 * n41;
    st.c20 = a20 + f02 * a22 + f04 * n42;
    st.c21 = a21 + f12 * a22 + f13 * n32 + f14 * n42;
    st.c22 = a22 + f24 * n42;
    st.c30 = n30;
    st.c31 = n31;
    st.c32 = n32;
    st.c40 = n40;
    st.c41 = n41;
    st.c42 = n42;
    return true;
}

// Two sequential scalar updates (y with sy2, then z with sz2); returns the chi2 increment.
// (ym, zm) is the measurement in the state's current (y, z) frame.  On return the frame has MOVED TO THE MEASUREMENT:
// st.y and st.z are relative to the attached hit, i.e. they hold the filtered residuals (-sigma^2/S * res, plus the
// z update's correction of y).  The model is translation invariant in y and z, so this is exact, and it keeps the
// magnitudes of st.y / st.z at the centimetre scale of one row step: without it a candidate that starts at
// z = 200 cm and is reported at z = 0 accumulates ~100 roundings of ulp(200 cm) in z (observed: 1.0e-4 cm on one
// tracklet in a million, the whole absolute tolerance).  The caller moves its reference (yref, zref) to the hit.
__device__ __forceinline__ float kf_update(KfState& st, float ym, float zm, float sy2, float sz2) {
    float chi2;
    {
        const float inv = rcp_ftz(st.c00 + sy2);
        const float res = ym - st.y;
        const float k1 = st.c10 * inv, k2 = st.c20 * inv, k3 = st.c30 * inv, k4 = st.c40 * inv;
        const float r = sy2 * inv;  // column 0 shrinks by sigma^2/S (no cancellation)
        chi2 = res * res * inv;
        st.y = -r * res;            // = y + K0 res - ym with K0 = 1 - sigma^2/S
        st.z = fmaf(k1, res, st.z);
        st.s = fmaf(k2, res, st.s);
        st.t = fmaf(k3, res, st.t);
        st.k = fmaf(k4, res, st.k);
        st.c11 = fmaf(-k1, st.c10, st.c11);
        st.c21 = fmaf(-k2, st.c10, st.c21);
        st.c22 = fmaf(-k2, st.c20, st.c22);
        st.c31 = fmaf(-k3, st.c10, st.c31);
        st.c32 = fmaf(-k3, st.c20, st.c32);
        st.c33 = fmaf(-k3, st.c30, st.c33);
        st.c41 = fmaf(-k4, st.c10, st.c41);
        st.c42 = fmaf(-k4, st.c20, st.c42);
        st.c43 = fmaf(-k4, st.c30, st.c43);
        st.c44 = fmaf(-k4, st.c40, st.c44);
        st.c00 *= r;
        st.c10 *= r;
        st.c20 *= r;
        st.c30 *= r;
        st.c40 *= r;
    }
    {
        const float inv = rcp_ftz(st.c11 + sz2);
        const float res = zm - st.z;
        const float k0 = st.c10 * inv, k2 = st.c21 * inv, k3 = st.c31 * inv, k4 = st.c41 * inv;
        const float r = sz2 * inv;
        chi2 = fmaf(res * res, inv, chi2);
        st.y = fmaf(k0, res, st.y);
        st.z = -r * res;
        st.s = fmaf(k2, res, st.s);
        st.t = fmaf(k3, res, st.t);
        st.k = fmaf(k4, res, st.k);
        st.c00 = fmaf(-k0, st.c10, st.c00);
        st.c20 = fmaf(-k2, st.c10, st.c20);
        st.c22 = fmaf(-k2, st.c21, st.c22);
        st.c30 = fmaf(-k3, st.c10, st.c30);
        st.c32 = fmaf(-k3, st.c21, st.c32);
        st.c33 = fmaf(-k3, st.c31, st.c33);
        st.c40 = fmaf(-k4, st.c10, st.c40);
        st.c42 = fmaf(-k4, st.c21, st.c42);
        st.c43 = fmaf(-k4, st.c31, st.c43);
        st.c44 = fmaf(-k4, st.c41, st.c44);
        st.c10 *= r;
        st.c11 *= r;
        st.c21 *= r;
        st.c31 *= r;
        st.c41 *= r;
    }
    return chi2;
}

// Change of sector frame (phase 2, reading M2): the state on the plane x of one sector-local frame becomes the state
// on the plane x1 of the frame rotated by +alpha about the beam axis (ca = cos alpha, sa = sin alpha).  y_abs is the
// ABSOLUTE y of the state (the kernels carry st.y relative to a reference); on return st.y is the absolute y in the
// new frame.  Exact rotation; the Jacobian of "state on the old plane -> state on the fixed new plane" has four
// non-trivial entries: sliding back to the plane along the track scales y by cos(phi)/cos(phi'), shifts z by the
// dz/ds of the slide and turns the direction by the curvature over it.  Returns false (state untouched) if
// |sinPhi| leaves [-max_s, max_s] or the rotated direction points backwards.
__device__ __forceinline__ bool kf_rotate(KfState& st, float y_abs, float x, float ca, float sa, float cB, float max_s,
                                          float& x1) {
    const float s = st.s;
    if (fabsf(s) > max_s) return false;
    const float c = sqrtf((1.0f - s) * (1.0f + s));
    const float s1 = s * ca - c * sa, c1 = c * ca + s * sa;
    if (fabsf(s1) > max_s || c1 <= 0.0f) return false;
    const float ic1 = 1.0f / c1;
    const float j00 = c * ic1, j10 = -sa * st.t * ic1, j20 = -sa * cB * st.k, j22 = c1 / c;
    x1 = x * ca + y_abs * sa;
    st.y = -x * sa + y_abs * ca;
    st.s = s1;
    // P <- J P J^T for rows y' = j00 y, z' = z + j10 y, s' = j20 y + j22 s (t, k unchanged)
    const float a20 = j20 * st.c00 + j22 * st.c20;  // cov(s', y)
    const float n11 = st.c11 + j10 * (2.0f * st.c10 + j10 * st.c00);
    const float n21 = j20 * st.c10 + j22 * st.c21 + j10 * a20;
    const float n22 = j20 * (j20 * st.c00 + 2.0f * j22 * st.c20) + j22 * j22 * st.c22;
    const float n31 = st.c31 + j10 * st.c30, n32 = j20 * st.c30 + j22 * st.c32;
    const float n41 = st.c41 + j10 * st.c40, n42 = j20 * st.c40 + j22 * st.c42;
    st.c10 = j00 * (st.c10 + j10 * st.c00);
    st.c00 = j00 * j00 * st.c00;
    st.c11 = n11;
    st.c20 = j00 * a20;
    st.c21 = n21;
    st.c22 = n22;
    st.c30 = j00 * st.c30;
    st.c31 = n31;
    st.c32 = n32;
    st.c40 = j00 * st.c40;
    st.c41 = n41;
    st.c42 = n42;
    return true;
}

// Seed: circle through three points in (x,y); dz/ds from the end points.  Returns false if |sinPhi| > max_s.
__device__ __forceinline__ bool kf_seed(KfState& st, float x0, float y0, float z0, float x1, float y1, float x2,
                                        float y2, float z2, float cB, float max_s, const float* p0) {
    const float ax = x1 - x0, ay = y1 - y0, bx = x2 - x0, by = y2 - y0;
    // The cross product cancels to ~1e-5 of its terms on a stiff track, and the seed's q/pt is the prior mean of a
    // weakly constrained parameter, so its rounding error would reach the fitted q/pt of short tracklets undiminished:
    // Kahan's difference of products (error <= 1.5 ulp of the result instead of ulp of the terms).
    const float w_ = ay * bx;
    const float cross = fmaf(ax, by, -w_) + fmaf(-ay, bx, w_);
    const float d01 = sqrtf(ax * ax + ay * ay), d02 = sqrtf(bx * bx + by * by);
    const float ex = x2 - x1, ey = y2 - y1;
    const float d12 = sqrtf(ex * ex + ey * ey);
    const float kap = 2.0f * cross / (d01 * d02 * d12);
    // sin(theta01 - asin(kappa d01 / 2)) expanded: sin A cos B - cos A sin B, with sin A = ay/d01, cos A = ax/d01
    const float sb = 0.5f * kap * d01;
    const float cb = sqrtf((1.0f - sb) * (1.0f + sb));
    const float sphi = (ay * cb - ax * sb) / d01;
    if (!(fabsf(sphi) <= max_s)) return false;
    const float S02 = d02 * asin_over(0.5f * kap * d02);
    st.y = y0;
    st.z = z0;
    st.s = sphi;
    st.t = (z2 - z0) / S02;
    st.k = cB != 0.0f ? kap / cB : 0.0f;
    st.c00 = p0[0]; st.c11 = p0[1]; st.c22 = p0[2]; st.c33 = p0[3]; st.c44 = p0[4];
    st.c10 = st.c20 = st.c21 = st.c30 = st.c31 = st.c32 = st.c40 = st.c41 = st.c42 = st.c43 = 0.0f;
    return true;
}

}  // namespace tpc
