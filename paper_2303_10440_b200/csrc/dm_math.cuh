// dm_math.cuh -- fp32 device arithmetic of the triangle Fourier integral (sm_100a).
//
//   f_T(k) = g(a,b,c) = iint_{t1,t2>=0, t1+t2<=1} exp(-i(a + t1 (b-a) + t2 (c-a))) dt1 dt2,   a = k.v1, b = k.v2, c = k.v3
//          = PAPER.md:162 eq. 9 / :194 eq. 14 (readings R1, R3) away from coincident arguments.
//
// Everything here works in the LOCAL form  g = e^{-ia} psi(p,q),  p = b-a = k.(v2-v1),  q = c-a = k.(v3-v1):
// the base phase a is reduced exactly (integer turns, see dm_phase_turns) and the gaps p, q come from fp32 edge
// vectors, so no gap is ever formed by subtracting two large phases ("sensitive to numerical
// precision").  psi is the second divided difference of exp on the nodes (0, -ip, -iq).
//
// Two evaluation branches cover every (p,q) (this is the "numerically stable branch" of north_star; the paper's
// eq. 15-16 are their zeroth-order limits, reading R4):
//   series   max(|p|,|q|,|q-p|) < DM_SERIES_RADIUS:  psi = sum_n (-i)^n h_n(p,q)/(n+2)!   (h_n complete homogeneous)
//   far-pair otherwise: psi = i (D(x_i,x_j) - D(x_j,x_k)) / (x_i - x_k) on the FARTHEST pair (x_i,x_k) of the nodes
//            {0,p,q}, with the first divided difference in its cancellation-free form
//            D(al,be) = exp[-i al, -i be] = e^{-i(al+be)/2} sinc((al-be)/2);  the only division is by a gap
//            >= DM_SERIES_RADIUS, so the absolute error stays O(1e-7 / DM_SERIES_RADIUS).
// The generic fast path (eq. 9 evaluated directly, used where its error bound allows) lives with the kernels.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define DM_SERIES_RADIUS 0.75f

struct cf {
    float re, im;
};
__device__ __forceinline__ cf cmul(cf a, cf b) { return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
__device__ __forceinline__ cf cscale(cf a, float s) { return {a.re * s, a.im * s}; }
__device__ __forceinline__ cf cadd(cf a, cf b) { return {a.re + b.re, a.im + b.im}; }
__device__ __forceinline__ cf csub(cf a, cf b) { return {a.re - b.re, a.im - b.im}; }
__device__ __forceinline__ cf cmul_i(cf a) { return {-a.im, a.re}; }  // i * a

// a b - c d with one rounding error of the result's own size (Kahan): exactly 0 when the two products are equal, so a
// triangle whose fp32 vertices are exactly collinear gets m_T = 0 exactly, as in the fp64 oracle (reading R19), and the
// normal of a thin triangle is as accurate as its fp32 edges allow.
__device__ __forceinline__ float dm_dop(float a, float b, float c, float d)
{
    const float w = __fmul_rn(c, d);
    const float e = __fmaf_rn(-c, d, w);
    const float f = __fmaf_rn(a, b, -w);
    return __fadd_rn(f, e);
}
// m = a x b
__device__ __forceinline__ void dm_cross(const float a[3], const float b[3], float m[3])
{
    m[0] = dm_dop(a[1], b[2], a[2], b[1]);
    m[1] = dm_dop(a[2], b[0], a[0], b[2]);
    m[2] = dm_dop(a[0], b[1], a[1], b[0]);
}

// sinc(h) = sin(h)/h and dsinc(h) = d/dh sinc = (cos h - sinc h)/h, without cancellation near 0.
__device__ __forceinline__ void dm_sinc_dsinc(float h, float& s, float& ds)
{
    const float h2 = h * h;
    if (fabsf(h) < 0.5f) {
        s = fmaf(h2, fmaf(h2, fmaf(h2, fmaf(h2, fmaf(h2, -1.0f / 39916800.0f, 1.0f / 362880.0f), -1.0f / 5040.0f),
                                   1.0f / 120.0f), -1.0f / 6.0f), 1.0f);
        ds = h * fmaf(h2, fmaf(h2, fmaf(h2, fmaf(h2, -1.0f / 3991680.0f, 1.0f / 45360.0f), -1.0f / 840.0f),
                               1.0f / 30.0f), -1.0f / 3.0f);
    } else {
        float sn, cs;
        sincosf(h, &sn, &cs);
        const float ih = 1.0f / h;
        s = sn * ih;
        ds = (cs - s) * ih;
    }
}

// First divided difference D(al,be) = exp[-i al, -i be] and (optionally) its partials.
//   dD/dal = e^{-im} ( ds/2 - i s/2 ),  dD/dbe = e^{-im} ( -ds/2 - i s/2 ),   m = (al+be)/2, h = (al-be)/2.
template <bool GRAD>
__device__ __forceinline__ void dm_dd2(float al, float be, cf& D, cf& dDa, cf& dDb)
{
    const float m = 0.5f * (al + be), h = 0.5f * (al - be);
    float s, ds, sn, cs;
    dm_sinc_dsinc(h, s, ds);
    sincosf(m, &sn, &cs);
    const cf e = {cs, -sn};
    D = cscale(e, s);
    if (GRAD) {
        dDa = cmul(e, cf{0.5f * ds, -0.5f * s});
        dDb = cmul(e, cf{-0.5f * ds, -0.5f * s});
    }
}

// Far-pair branch on nodes (x_i, x_j, x_k), (x_i,x_k) the farthest pair.
//   psi = i (D_ij - D_jk)/d,  d = x_i - x_k
//   dpsi/dx_j = i (dD_ij/dbe - dD_jk/dal)/d
//   dpsi/dx_i = i dD_ij/dal / d - psi/d          dpsi/dx_k = -i dD_jk/dbe / d + psi/d
template <bool GRAD>
__device__ __forceinline__ void dm_psi_far(float xi, float xj, float xk, cf& psi, cf& di, cf& dj, cf& dk)
{
    const float invd = 1.0f / (xi - xk);
    cf D1, D1a, D1b, D2, D2a, D2b;
    dm_dd2<GRAD>(xi, xj, D1, D1a, D1b);
    dm_dd2<GRAD>(xj, xk, D2, D2a, D2b);
    psi = cscale(cmul_i(csub(D1, D2)), invd);
    if (GRAD) {
        dj = cscale(cmul_i(csub(D1b, D2a)), invd);
        di = cscale(csub(cmul_i(D1a), psi), invd);
        dk = cscale(csub(psi, cmul_i(D2b)), invd);
    }
}

// Series branch: psi = sum_n (-i)^n h_n(p,q)/(n+2)!,
//   dpsi/dp = -i exp[0,-ip,-ip,-iq] = -i sum_n (-i)^n h_n(p,p,q)/(n+3)!,  likewise dq with h_n(p,q,q);
//   h_n(p,q) = p h_{n-1}(p,q) + q^n,  h_n(p,p,q) = p h_{n-1}(p,p,q) + h_n(p,q),  h_n(p,q,q) = q h_{n-1}(p,q,q) + h_n(p,q).
// 10 terms: the first dropped term is below 2e-9 for max gap < 0.75.
template <bool GRAD>
__device__ __forceinline__ void dm_psi_series(float p, float q, cf& psi, cf& dp, cf& dq)
{
    // 1/(n+2)! and 1/(n+3)! for n = 0..9
    const float f2[10] = {1.0f / 2, 1.0f / 6, 1.0f / 24, 1.0f / 120, 1.0f / 720, 1.0f / 5040, 1.0f / 40320,
                          1.0f / 362880, 1.0f / 3628800, 1.0f / 39916800};
    const float f3[10] = {1.0f / 6, 1.0f / 24, 1.0f / 120, 1.0f / 720, 1.0f / 5040, 1.0f / 40320, 1.0f / 362880,
                          1.0f / 3628800, 1.0f / 39916800, 1.0f / 479001600};
    float qn = 1.0f, h2 = 1.0f, hp = 1.0f, hq = 1.0f;  // q^n, h_n(p,q), h_n(p,p,q), h_n(p,q,q) at n = 0
    float s_re = 0.f, s_im = 0.f, p_re = 0.f, p_im = 0.f, q_re = 0.f, q_im = 0.f;
#pragma unroll
    for (int n = 0; n < 10; ++n) {
        if (n > 0) {
            qn *= q;
            h2 = fmaf(p, h2, qn);
            if (GRAD) {
                hp = fmaf(p, hp, h2);
                hq = fmaf(q, hq, h2);
            }
        }
        // (-i)^n: n%4 = 0: +1, 1: -i, 2: -1, 3: +i
        const float sg = (n & 2) ? -1.0f : 1.0f;
        if ((n & 1) == 0) {
            s_re = fmaf(sg * f2[n], h2, s_re);
            if (GRAD) {
                p_re = fmaf(sg * f3[n], hp, p_re);
                q_re = fmaf(sg * f3[n], hq, q_re);
            }
        } else {
            s_im = fmaf(-sg * f2[n], h2, s_im);
            if (GRAD) {
                p_im = fmaf(-sg * f3[n], hp, p_im);
                q_im = fmaf(-sg * f3[n], hq, q_im);
            }
        }
    }
    psi = {s_re, s_im};
    if (GRAD) {
        dp = {p_im, -p_re};  // -i * (p_re + i p_im)
        dq = {q_im, -q_re};
    }
}

// ---- branch-free ("pooled") variant of the far-pair branch -------------------------------------------------------------
// Used for the flagged pairs of the fast backward kernel, where the 32 lanes of a warp hold UNRELATED pairs: every lane
// runs the same instructions (roles are chosen by selects, sinc by select between polynomial and MUFU quotient), and the
// sines / cosines are MUFU approximations on arguments reduced to [-pi, pi] (abs. error ~5e-7; these pairs are a few per
// cent of all pairs and need ~1e-5).  Requires max gap >= DM_SERIES_RADIUS.
__device__ __forceinline__ float dm_rcp_approx(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ void dm_sinc_dsinc_uniform(float h, float& s, float& ds)
{
    const float h2 = h * h;
    const float sp = fmaf(h2, fmaf(h2, fmaf(h2, fmaf(h2, fmaf(h2, -1.0f / 39916800.0f, 1.0f / 362880.0f), -1.0f / 5040.0f),
                                            1.0f / 120.0f), -1.0f / 6.0f), 1.0f);
    const float dsp = h * fmaf(h2, fmaf(h2, fmaf(h2, fmaf(h2, -1.0f / 3991680.0f, 1.0f / 45360.0f), -1.0f / 840.0f),
                                        1.0f / 30.0f), -1.0f / 3.0f);
    const float hr = fmaf(-6.283185307179586f, rintf(h * 0.15915494309189535f), h);
    const float sn = __sinf(hr), cs = __cosf(hr);
    const float ih = dm_rcp_approx(h);
    const float sb = sn * ih, dsb = (cs - sb) * ih;
    const bool small = fabsf(h) < 0.5f;
    s = small ? sp : sb;
    ds = small ? dsp : dsb;
}
__device__ __forceinline__ void dm_dd2_uniform(float al, float be, cf& D, cf& dDa, cf& dDb)
{
    const float m = 0.5f * (al + be), h = 0.5f * (al - be);
    float s, ds;
    dm_sinc_dsinc_uniform(h, s, ds);
    const float mr = fmaf(-6.283185307179586f, rintf(m * 0.15915494309189535f), m);
    const cf e = {__cosf(mr), -__sinf(mr)};
    D = cscale(e, s);
    dDa = cmul(e, cf{0.5f * ds, -0.5f * s});
    dDb = cmul(e, cf{-0.5f * ds, -0.5f * s});
}
// psi(p,q), dpsi/dp, dpsi/dq on nodes (0, p, q) with max gap >= DM_SERIES_RADIUS; same formulas as dm_psi_far
__device__ __forceinline__ void dm_psi_far_uniform(float p, float q, cf& psi, cf& dp, cf& dq)
{
    const float ap = fabsf(p), aq = fabsf(q), ar = fabsf(q - p);
    const bool A = (aq >= ap && aq >= ar);   // pair (0,2): i=0, j=1, k=2
    const bool B = !A && (ap >= ar);         // pair (0,1): i=0, j=2, k=1;  else pair (1,2): i=1, j=0, k=2
    const float xi = (A || B) ? 0.0f : p;
    const float xj = A ? p : (B ? q : 0.0f);
    const float xk = B ? p : q;
    const float invd = dm_rcp_approx(xi - xk);
    cf D1, D1a, D1b, D2, D2a, D2b;
    dm_dd2_uniform(xi, xj, D1, D1a, D1b);
    dm_dd2_uniform(xj, xk, D2, D2a, D2b);
    psi = cscale(cmul_i(csub(D1, D2)), invd);
    const cf dj = cscale(cmul_i(csub(D1b, D2a)), invd);
    const cf di = cscale(csub(cmul_i(D1a), psi), invd);
    const cf dk = cscale(csub(psi, cmul_i(D2b)), invd);
    // node 1 is j (A), k (B) or i (C); node 2 is k (A), j (B) or k (C)
    dp.re = A ? dj.re : (B ? dk.re : di.re);
    dp.im = A ? dj.im : (B ? dk.im : di.im);
    dq.re = B ? dj.re : dk.re;
    dq.im = B ? dj.im : dk.im;
}

// psi(p,q) alone, any (p,q), with MUFU sines / cosines on arguments reduced to [-pi, pi] (abs. error ~5e-7) -- for the
// flagged pairs of the fast forward kernel: each is one triangle's term among >= 10^2..10^5, needed to ~1e-5 of its own size
// (DESIGN.md section 6), and the fast path's own phase seeds have the same accuracy.  Same two branches as dm_psi_robust.
__device__ __forceinline__ cf dm_dd2_value_fast(float al, float be)
{
    const float m = 0.5f * (al + be), h = 0.5f * (al - be);
    float s;
    if (fabsf(h) < 0.5f) {
        const float h2 = h * h;
        s = fmaf(h2, fmaf(h2, fmaf(h2, fmaf(h2, fmaf(h2, -1.0f / 39916800.0f, 1.0f / 362880.0f), -1.0f / 5040.0f), 1.0f / 120.0f),
                          -1.0f / 6.0f), 1.0f);
    } else {
        const float hr = fmaf(-6.283185307179586f, rintf(h * 0.15915494309189535f), h);
        s = __sinf(hr) * dm_rcp_approx(h);
    }
    const float mr = fmaf(-6.283185307179586f, rintf(m * 0.15915494309189535f), m);
    return {__cosf(mr) * s, -__sinf(mr) * s};
}
__device__ __forceinline__ cf dm_psi_value_fast(float p, float q)
{
    const float ap = fabsf(p), aq = fabsf(q), ar = fabsf(q - p);
    if (fmaxf(fmaxf(ap, aq), ar) < DM_SERIES_RADIUS) {
        cf psi, d1, d2;
        dm_psi_series<false>(p, q, psi, d1, d2);
        return psi;
    }
    // nodes x0 = 0, x1 = p, x2 = q; the farthest pair (x_i, x_k) decides the roles, x_j is the third node
    const bool A = (aq >= ap && aq >= ar);   // pair (0,2): i=0, j=1, k=2
    const bool B = !A && (ap >= ar);         // pair (0,1): i=0, j=2, k=1;  else pair (1,2): i=1, j=0, k=2
    const float xi = (A || B) ? 0.0f : p;
    const float xj = A ? p : (B ? q : 0.0f);
    const float xk = B ? p : q;
    const cf D1 = dm_dd2_value_fast(xi, xj), D2 = dm_dd2_value_fast(xj, xk);
    return cscale(cmul_i(csub(D1, D2)), dm_rcp_approx(xi - xk));
}

// psi(p,q) and its partials, any (p,q).  Robust ("slow") path.
template <bool GRAD>
__device__ __forceinline__ void dm_psi_robust(float p, float q, cf& psi, cf& dp, cf& dq)
{
    const float r = q - p;
    const float ap = fabsf(p), aq = fabsf(q), ar = fabsf(r);
    if (fmaxf(fmaxf(ap, aq), ar) < DM_SERIES_RADIUS) {
        dm_psi_series<GRAD>(p, q, psi, dp, dq);
        return;
    }
    // nodes x0 = 0, x1 = p, x2 = q; farthest pair decides the roles (i, j, k)
    cf d0, d1, d2;
    if (aq >= ap && aq >= ar) {          // pair (0,2): i=0, j=1, k=2
        dm_psi_far<GRAD>(0.0f, p, q, psi, d0, d1, d2);
    } else if (ap >= ar) {               // pair (0,1): i=0, j=2, k=1
        dm_psi_far<GRAD>(0.0f, q, p, psi, d0, d2, d1);
    } else {                             // pair (1,2): i=1, j=0, k=2
        dm_psi_far<GRAD>(p, 0.0f, q, psi, d1, d0, d2);
    }
    if (GRAD) {
        dp = d1;
        dq = d2;
    }
}

// Exact base phase.  Vertex coordinates are stored as unsigned 32-bit fixed-point TURNS u = frac(v_a / L_a);
// the grid frequencies are integer multiples of 2 pi / L_a, so  k.v / (2 pi) = n_x u_x + n_y u_y + n_z u_z
// (mod 1) is computed exactly by wrapping 32-bit integer arithmetic.  Returns e^{-i k.v}.
__device__ __forceinline__ uint32_t dm_phase_turns(int nx, int ny, int nz, uint32_t ux, uint32_t uy, uint32_t uz)
{
    return (uint32_t)nx * ux + (uint32_t)ny * uy + (uint32_t)nz * uz;
}
// fast e^{-2 pi i t} from integer turns: MUFU sin/cos on an argument reduced exactly to [-pi, pi)
__device__ __forceinline__ cf dm_expmi_turns_fast(uint32_t turns)
{
    const float x = (float)(int32_t)turns * (6.283185307179586f / 4294967296.0f);
    return {__cosf(x), -__sinf(x)};
}
__device__ __forceinline__ cf dm_expmi_turns(uint32_t turns)
{
    const float t = (float)(int32_t)turns * (1.0f / 2147483648.0f);  // 2*turns in [-1, 1)
    float sn, cs;
    sincospif(t, &sn, &cs);
    return {cs, -sn};
}
