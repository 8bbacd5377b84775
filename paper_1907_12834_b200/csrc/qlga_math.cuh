// qlga_math.cuh -- per-site device arithmetic of the spin-2 QLGA step (sm_100a).
//
// Everything here works on one lattice site held in registers:
//   * kinetic messages of I'_{d,sigma} = S C S^T C (eq. 107)
//     written as a radius-1 stencil,
//   * the interaction unitary U^{(s)} = exp(-i s H_int[psi]) (reading R4,
//     eq. 34) as scalar phase x Horner polynomial of
//     K = c1 F.f + (c2/5)|chi><chi| applied to the two spinor 5-vectors.
// No code is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace qlga {

template <typename T> struct vec2;
template <> struct vec2<double> { using type = double2; };
template <> struct vec2<float>  { using type = float2; };

template <typename T> struct cx {
    T re, im;
};

template <typename T> __device__ __forceinline__ cx<T> mk(T re, T im) { cx<T> z; z.re = re; z.im = im; return z; }
template <typename T> __device__ __forceinline__ cx<T> operator+(cx<T> a, cx<T> b) { return mk<T>(a.re + b.re, a.im + b.im); }
template <typename T> __device__ __forceinline__ cx<T> operator-(cx<T> a, cx<T> b) { return mk<T>(a.re - b.re, a.im - b.im); }
template <typename T> __device__ __forceinline__ cx<T> cmul(cx<T> a, cx<T> b) {
    return mk<T>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re);
}
// acc + a*b
template <typename T> __device__ __forceinline__ cx<T> cfma(cx<T> a, cx<T> b, cx<T> acc) {
    acc.re = fma(a.re, b.re, acc.re); acc.re = fma(-a.im, b.im, acc.re);
    acc.im = fma(a.re, b.im, acc.im); acc.im = fma(a.im, b.re, acc.im);
    return acc;
}
// acc + conj(a)*b
template <typename T> __device__ __forceinline__ cx<T> cfma_conj(cx<T> a, cx<T> b, cx<T> acc) {
    acc.re = fma(a.re, b.re, acc.re); acc.re = fma(a.im, b.im, acc.re);
    acc.im = fma(a.re, b.im, acc.im); acc.im = fma(-a.im, b.re, acc.im);
    return acc;
}

// sin/cos of the scalar interaction phase for |x| <= 2^-4 (always the case at the
// paper's scaled amplitudes): Taylor polynomials in x^2 to x^13 / x^14, remainder
// < 2^-80, branch free so that the chain interleaves with the spin-density arithmetic.
template <typename T>
__device__ __forceinline__ void sincos_small(T x, T* s, T* c) {
    const T z = x * x;
    T ps = fma(z, (T)(-1.0 / 156.0), (T)1);
    T pc = fma(z, (T)(-1.0 / 182.0), (T)1);
    ps = fma(z * (T)(-1.0 / 110.0), ps, (T)1);
    pc = fma(z * (T)(-1.0 / 132.0), pc, (T)1);
    ps = fma(z * (T)(-1.0 / 72.0), ps, (T)1);
    pc = fma(z * (T)(-1.0 / 90.0), pc, (T)1);
    ps = fma(z * (T)(-1.0 / 42.0), ps, (T)1);
    pc = fma(z * (T)(-1.0 / 56.0), pc, (T)1);
    ps = fma(z * (T)(-1.0 / 20.0), ps, (T)1);
    pc = fma(z * (T)(-1.0 / 30.0), pc, (T)1);
    ps = fma(z * (T)(-1.0 / 6.0), ps, (T)1);
    pc = fma(z * (T)(-1.0 / 12.0), pc, (T)1);
    *s = x * ps;
    *c = fma(z * (T)-0.5, pc, (T)1);
}
__device__ __forceinline__ void sincos_lib(double x, double* s, double* c) { sincos(x, s, c); }
__device__ __forceinline__ void sincos_lib(float x, float* s, float* c) { sincosf(x, s, c); }

// Site state: q[j][sigma], j = 0..4 <-> m = +2..-2.
template <typename T> struct Site {
    cx<T> q[5][2];
};

// ---------------------------------------------------------------------------
// Kinetic factor I'_{d,sigma} as a stencil, halvings deferred.
// With a = streamed component sigma, b = the other one:
//   Fw = i a + b   (goes to the site at r + e)      Bw = a + i b   (goes to r - e)
//   a'(r) = -i Bw(r) + Fw(r - e)                    b'(r) = -i Fw(r) + Bw(r + e)
// and the true result is (a', b')/2; the caller folds the power of two into the
// interaction constants and into one final scaling (exact in binary floating point).
// ---------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ void kin_messages(const Site<T>& s, int sigma, cx<T> Fw[5], cx<T> Bw[5]) {
#pragma unroll
    for (int j = 0; j < 5; ++j) {
        cx<T> a = s.q[j][sigma], b = s.q[j][1 - sigma];
        Fw[j] = mk<T>(b.re - a.im, b.im + a.re);
        Bw[j] = mk<T>(a.re - b.im, a.im + b.re);
    }
}

template <typename T>
__device__ __forceinline__ void kin_update(Site<T>& s, int sigma, const cx<T> Fw[5], const cx<T> Bw[5],
                                           const cx<T> Fprev[5], const cx<T> Bnext[5]) {
#pragma unroll
    for (int j = 0; j < 5; ++j) {
        s.q[j][sigma]     = mk<T>(Fprev[j].re + Bw[j].im, Fprev[j].im - Bw[j].re);
        s.q[j][1 - sigma] = mk<T>(Bnext[j].re + Fw[j].im, Bnext[j].im - Fw[j].re);
    }
}

// ---------------------------------------------------------------------------
// Interaction.  Constants of one application (already multiplied by the
// sub-step fraction s and by the deferred-scaling factor 4^-e):
//   g0 = s c0, g1 = s c1, g2 = s c2 / 5.
// thr[p-1] = largest angle for which a degree-p polynomial meets the tolerance.
// ---------------------------------------------------------------------------
constexpr int QLGA_PMAX = 12;

template <typename T> struct UConst {
    T g0, g1, g2;
};

struct ExpTable {
    // Horner ratios of the degree-p polynomial P_p(y) = b0 (1 + r1 y (1 + r2 y (... (1 + rp y)))),
    // y = -i s K: r[p-1][k] = b_k / b_{k-1} (close to 1/k), b0[p-1] close to 1.  P_p is the
    // Chebyshev-economised Taylor polynomial of exp(y) on |y| <= thr[p-1].
    double r[QLGA_PMAX][QLGA_PMAX + 1];
    double b0[QLGA_PMAX];
    float thr[QLGA_PMAX];       // thr[p-1] = largest angle degree p serves within the tolerance
    float theta_split;          // angles above this are split into equal sub-angles
};

// w = (s K) u  with  s K = g1 F.f + g2 |chi><chi|,
//   (F.f u)_m = m F_z u_m + (1/2) F_- alpha_{m-1} u_{m-1} + (1/2) F_+ alpha_m u_{m+1},
//   alpha_1 = alpha_-2 = 2, alpha_0 = alpha_-1 = sqrt(6)   (f_+|m> = sqrt(6 - m(m+1))|m+1>),
//   <chi|u> = sum_m (-1)^m psi_{-m} u_m,   chi_m = (-1)^m conj(psi_{-m}).
// Inputs are pre-scaled: az = g1 F_z, a1 = g1 F_+ (coefficient 2/2), a6 = g1 (sqrt6/2) F_+.
template <typename T>
__device__ __forceinline__ void apply_sK(const cx<T> u[5], cx<T> w[5], T az, cx<T> a1, cx<T> a6,
                                         T g2, const cx<T> psi[5]) {
    // rank-one part: t = g2 <chi|u>
    cx<T> t = cmul(psi[4], u[0]);
    t = cfma(psi[2], u[2], t);
    t = cfma(psi[0], u[4], t);
    cx<T> t2 = cmul(psi[3], u[1]);
    t2 = cfma(psi[1], u[3], t2);
    t = t - t2;
    t.re *= g2; t.im *= g2;
    // spin part, rows m = +2..-2 (j = 0..4); raising uses conj(F_+) on u_{m-1} (j+1),
    // lowering uses F_+ on u_{m+1} (j-1)
    const T two = (T)2;
    cx<T> r0 = mk<T>(two * az * u[0].re, two * az * u[0].im);
    r0 = cfma_conj(a1, u[1], r0);
    cx<T> r1 = mk<T>(az * u[1].re, az * u[1].im);
    r1 = cfma(a1, u[0], r1);
    r1 = cfma_conj(a6, u[2], r1);
    cx<T> r2 = cmul(a6, u[1]);
    r2 = cfma_conj(a6, u[3], r2);
    cx<T> r3 = mk<T>(-az * u[3].re, -az * u[3].im);
    r3 = cfma(a6, u[2], r3);
    r3 = cfma_conj(a1, u[4], r3);
    cx<T> r4 = mk<T>(-two * az * u[4].re, -two * az * u[4].im);
    r4 = cfma(a1, u[3], r4);
    // add t * chi_m,  chi_m = (-1)^m conj(psi_{-m})
    w[0] = cfma_conj(psi[4], t, r0);
    w[1] = r1 - cfma_conj(psi[3], t, mk<T>((T)0, (T)0));
    w[2] = cfma_conj(psi[2], t, r2);
    w[3] = r3 - cfma_conj(psi[1], t, mk<T>((T)0, (T)0));
    w[4] = cfma_conj(psi[0], t, r4);
}

// number of thresholds thr[0..PMAX-2] (ascending) that theta exceeds: independent
// compares summed as a tree (a bisection has fewer instructions but is a chain of
// dependent constant-bank loads, and this sits on the critical path of every factor)
__device__ __forceinline__ int count_below(const float* thr, float theta) {
    int c[QLGA_PMAX - 1];
#pragma unroll
    for (int k = 0; k < QLGA_PMAX - 1; ++k) c[k] = (theta > thr[k]) ? 1 : 0;
#pragma unroll
    for (int w = 1; w < QLGA_PMAX - 1; w *= 2)
#pragma unroll
        for (int k = 0; k + w < QLGA_PMAX - 1; k += 2 * w) c[k] += c[k + w];
    return c[0];
}

// Site-local coefficients of sK = g1 F.f + g2 |chi><chi| (pre-scaled, see apply_sK).
template <typename T> struct KCoef {
    T az, g2;
    cx<T> a1, a6;
    cx<T> psi[5];
    T rho;
    float theta;                                   // 2|g1||F| + |g2| rho, this lane
};

template <typename T>
__device__ __forceinline__ void site_coefficients(const Site<T>& s, const UConst<T>& uc, KCoef<T>& kc) {
    T n[5];
#pragma unroll
    for (int j = 0; j < 5; ++j) {
        kc.psi[j] = s.q[j][0] + s.q[j][1];
        n[j] = fma(kc.psi[j].re, kc.psi[j].re, kc.psi[j].im * kc.psi[j].im);
    }
    kc.rho = (n[0] + n[4]) + (n[1] + n[3]) + n[2];
    const T Fz = (T)2 * (n[0] - n[4]) + (n[1] - n[3]);
    // F_+ = sum_m alpha_m conj(psi_{m+1}) psi_m = 2(conj(psi_2) psi_1 + conj(psi_-1) psi_-2)
    //                                           + sqrt6 (conj(psi_1) psi_0 + conj(psi_0) psi_-1)
    cx<T> fa = cfma_conj(kc.psi[0], kc.psi[1], mk<T>((T)0, (T)0));
    fa = cfma_conj(kc.psi[3], kc.psi[4], fa);
    cx<T> fb = cfma_conj(kc.psi[1], kc.psi[2], mk<T>((T)0, (T)0));
    fb = cfma_conj(kc.psi[2], kc.psi[3], fb);
    const T rt6 = (T)2.4494897427831780981972840747059;
    const cx<T> Fp = mk<T>(fma(rt6, fb.re, (T)2 * fa.re), fma(rt6, fb.im, (T)2 * fa.im));
    // angle bound theta = 2 |g1| |F| + |g2| rho (the exact spectral norms of the two parts);
    // |F| by the approximate reciprocal square root (2 ulp; the 2^-10 margin covers it)
    const float f2 = fmaxf((float)(Fz * Fz + Fp.re * Fp.re + Fp.im * Fp.im), 1e-37f);
    const float Fabs = f2 * __frsqrt_rn(f2);
    kc.theta = (2.0f * fabsf((float)uc.g1) * Fabs + fabsf((float)uc.g2) * (float)kc.rho) * 1.0009765625f;
    kc.g2 = uc.g2;
    kc.az = uc.g1 * Fz;
    kc.a1 = mk<T>(uc.g1 * Fp.re, uc.g1 * Fp.im);
    const T rt6h = (T)1.2247448713915890490986420373529;          // sqrt(6)/2
    kc.a6 = mk<T>(rt6h * kc.a1.re, rt6h * kc.a1.im);
}

// u <- P_p(-i sK) v in Horner form u_{k-1} = v + r_k (-i sK) u_k, k = p..1, u_p = v
// (stage p acts on v itself: no copy).  psi, hence K, is frozen (reading R4).
template <typename T>
__device__ __forceinline__ void horner(const cx<T> v[5], cx<T> u[5], const KCoef<T>& kc,
                                       const double* __restrict__ r, int p) {
    cx<T> w[5];
    apply_sK<T>(v, w, kc.az, kc.a1, kc.a6, kc.g2, kc.psi);
    {
        const T ik = (T)r[p];
#pragma unroll
        for (int j = 0; j < 5; ++j) {
            u[j].re = fma(ik, w[j].im, v[j].re); u[j].im = fma(-ik, w[j].re, v[j].im);
        }
    }
#pragma unroll 1
    for (int k = p - 1; k >= 1; --k) {
        apply_sK<T>(u, w, kc.az, kc.a1, kc.a6, kc.g2, kc.psi);
        const T ik = (T)r[k];
#pragma unroll
        for (int j = 0; j < 5; ++j) {
            u[j].re = fma(ik, w[j].im, v[j].re); u[j].im = fma(-ik, w[j].re, v[j].im);
        }
    }
}

// General path (never taken at the paper's amplitudes): scalar phase by the library
// sincos; angles above theta_split in nsub equal sub-angles (exact: K is frozen).
// Out of line and by value so that the common path keeps its registers.
template <typename T>
__device__ __noinline__ Site<T> interaction_general(Site<T> s, UConst<T> uc, const ExpTable& tab, float theta) {
    KCoef<T> kc;
    site_coefficients<T>(s, uc, kc);
    int nsub = 1;
    if (theta > tab.theta_split) nsub = (int)ceilf(theta / tab.theta_split);
    const T inv_nsub = (T)1 / (T)nsub;
    kc.g2 *= inv_nsub; kc.az *= inv_nsub;
    kc.a1.re *= inv_nsub; kc.a1.im *= inv_nsub; kc.a6.re *= inv_nsub; kc.a6.im *= inv_nsub;
    const int p = 1 + count_below(tab.thr, theta / (float)nsub * 1.0009765625f);
    T sn, cs;
    sincos_lib(uc.g0 * kc.rho, &sn, &cs);
    T b0n = (T)1;
    for (int rep = 0; rep < nsub; ++rep) b0n *= (T)tab.b0[p - 1];
    const cx<T> ph = mk<T>(b0n * cs, -(b0n * sn));
    for (int sg = 0; sg < 2; ++sg) {
        cx<T> v[5], u[5];
        for (int j = 0; j < 5; ++j) v[j] = s.q[j][sg];
        for (int rep = 0; rep < nsub; ++rep) {
            horner<T>(v, u, kc, tab.r[p - 1], p);
            for (int j = 0; j < 5; ++j) v[j] = u[j];
        }
        for (int j = 0; j < 5; ++j) s.q[j][sg] = cmul(ph, v[j]);
    }
    return s;
}

// Apply U^{(s)} to one site.  The site may carry a power-of-two scale 2^e; the
// caller passes constants multiplied by 4^-e, which makes the result identical
// (bit for bit, barring under/overflow) to applying U to the unscaled site.
template <typename T>
__device__ __forceinline__ void interaction(Site<T>& s, const UConst<T>& uc, const ExpTable& tab) {
    KCoef<T> kc;
    site_coefficients<T>(s, uc, kc);
    // The first Horner stage of component 1 needs neither the degree nor the phase: it is
    // issued before the warp-wide reductions below so that their latency (rsqrt, REDUX,
    // vote, the branch on their result) is covered by 88 independent FP64 instructions.
    cx<T> va[5], wa[5];
#pragma unroll
    for (int j = 0; j < 5; ++j) va[j] = s.q[j][0];
    apply_sK<T>(va, wa, kc.az, kc.a1, kc.a6, kc.g2, kc.psi);
    // warp-uniform angle (one polynomial degree per warp keeps the Horner loops convergent)
    const float theta = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(kc.theta)));
    const T xph = uc.g0 * kc.rho;                  // scalar phase exp(-i s c0 rho)
    const bool big_phase = !__all_sync(0xffffffffu, fabs(xph) <= (T)0.0625);
    if (big_phase || theta > tab.theta_split) {
        s = interaction_general<T>(s, uc, tab, theta);
        return;
    }
    T sn, cs;
    sincos_small<T>(xph, &sn, &cs);
    const int p = 1 + count_below(tab.thr, theta);
    const T pb0 = (T)tab.b0[p - 1];                // constant term of the polynomial (1 - O(tol))
    const cx<T> ph = mk<T>(pb0 * cs, -(pb0 * sn));
    const double* r = tab.r[p - 1];
    {
        cx<T> u[5];
        const T ik = (T)r[p];
#pragma unroll
        for (int j = 0; j < 5; ++j) {
            u[j].re = fma(ik, wa[j].im, va[j].re); u[j].im = fma(-ik, wa[j].re, va[j].im);
        }
#pragma unroll 1
        for (int k = p - 1; k >= 1; --k) {
            apply_sK<T>(u, wa, kc.az, kc.a1, kc.a6, kc.g2, kc.psi);
            const T ikk = (T)r[k];
#pragma unroll
            for (int j = 0; j < 5; ++j) {
                u[j].re = fma(ikk, wa[j].im, va[j].re); u[j].im = fma(-ikk, wa[j].re, va[j].im);
            }
        }
#pragma unroll
        for (int j = 0; j < 5; ++j) s.q[j][0] = cmul(ph, u[j]);
    }
    {
        cx<T> v[5], u[5];
#pragma unroll
        for (int j = 0; j < 5; ++j) v[j] = s.q[j][1];
        horner<T>(v, u, kc, r, p);
#pragma unroll
        for (int j = 0; j < 5; ++j) s.q[j][1] = cmul(ph, u[j]);
    }
}

}  // namespace qlga
