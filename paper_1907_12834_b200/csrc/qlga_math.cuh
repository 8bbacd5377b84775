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
#include <math.h>

namespace qlga {

template <typename T> struct vec2;
template <> struct vec2<double> { using type = double2; };
template <> struct vec2<float>  { using type = float2; };

template <typename T> struct __align__(2 * sizeof(T)) cx {   // one 16-byte / 8-byte element, as in memory
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

// acc - conj(a)*b
template <typename T> __device__ __forceinline__ cx<T> cfnma_conj(cx<T> a, cx<T> b, cx<T> acc) {
    acc.re = fma(-a.re, b.re, acc.re); acc.re = fma(-a.im, b.im, acc.re);
    acc.im = fma(-a.re, b.im, acc.im); acc.im = fma(a.im, b.re, acc.im);
    return acc;
}
// a * conj(b)
template <typename T> __device__ __forceinline__ cx<T> cmul_conj(cx<T> a, cx<T> b) {
    return mk<T>(fma(a.re, b.re, a.im * b.im), fma(a.im, b.re, -(a.re * b.im)));
}

// real * complex, acc + real * complex
template <typename T> __device__ __forceinline__ cx<T> rmul(T a, cx<T> u) { return mk<T>(a * u.re, a * u.im); }
template <typename T> __device__ __forceinline__ cx<T> rfma(T a, cx<T> u, cx<T> acc) {
    return mk<T>(fma(a, u.re, acc.re), fma(a, u.im, acc.im));
}
// a + i b,  a - i b,  v - i k w  (multiplication by +-i is a swap with one sign change)
template <typename T> __device__ __forceinline__ cx<T> add_i(cx<T> a, cx<T> b) { return mk<T>(a.re - b.im, a.im + b.re); }
template <typename T> __device__ __forceinline__ cx<T> sub_i(cx<T> a, cx<T> b) { return mk<T>(a.re + b.im, a.im - b.re); }
template <typename T> __device__ __forceinline__ cx<T> axmi(T k, cx<T> w, cx<T> v) {
    return mk<T>(fma(k, w.im, v.re), fma(-k, w.re, v.im));
}

// ---------------------------------------------------------------------------
// fp32: packed arithmetic.  sm_100a has two-wide fp32 instructions (FFMA2, FADD2, FMUL2:
// fma.rn.f32x2 ...) whose operands take a scalar broadcast, a half swap and per-half signs
// as free modifiers, so a complex number held as one (re, im) register pair costs one
// instruction per real-complex product or addition and two per complex-complex product:
// half the issue slots of the scalar form.  Non-template overloads for cx<float>; the
// fp64 path keeps the generic templates above (there is no packed fp64 arithmetic).
// ---------------------------------------------------------------------------
__device__ __forceinline__ float2 pk(cx<float> z) { return make_float2(z.re, z.im); }
__device__ __forceinline__ float2 pk_i(cx<float> z) { return make_float2(-z.im, z.re); }     // i z
__device__ __forceinline__ float2 pk_mi(cx<float> z) { return make_float2(z.im, -z.re); }    // -i z
__device__ __forceinline__ float2 bc(float a) { return make_float2(a, a); }
__device__ __forceinline__ cx<float> up(float2 v) { return mk<float>(v.x, v.y); }
__device__ __forceinline__ cx<float> operator+(cx<float> a, cx<float> b) { return up(__fadd2_rn(pk(a), pk(b))); }
__device__ __forceinline__ cx<float> operator-(cx<float> a, cx<float> b) {
    return up(__fadd2_rn(pk(a), make_float2(-b.re, -b.im)));
}
// (the swap / sign modifiers exist on the first source operand of FFMA2 / FMUL2, the scalar
// broadcast on the second: the complex value goes first, the broadcast coefficient second)
__device__ __forceinline__ cx<float> cmul(cx<float> a, cx<float> b) {
    return up(__ffma2_rn(pk_i(b), bc(a.im), __fmul2_rn(pk(b), bc(a.re))));
}
__device__ __forceinline__ cx<float> cfma(cx<float> a, cx<float> b, cx<float> acc) {
    return up(__ffma2_rn(pk_i(b), bc(a.im), __ffma2_rn(pk(b), bc(a.re), pk(acc))));
}
__device__ __forceinline__ cx<float> cfma_conj(cx<float> a, cx<float> b, cx<float> acc) {
    return up(__ffma2_rn(pk_mi(b), bc(a.im), __ffma2_rn(pk(b), bc(a.re), pk(acc))));
}
__device__ __forceinline__ cx<float> cfnma_conj(cx<float> a, cx<float> b, cx<float> acc) {
    return up(__ffma2_rn(pk_i(b), bc(a.im), __ffma2_rn(pk(b), bc(-a.re), pk(acc))));
}
__device__ __forceinline__ cx<float> cmul_conj(cx<float> a, cx<float> b) {
    return up(__ffma2_rn(pk_mi(a), bc(b.im), __fmul2_rn(pk(a), bc(b.re))));
}
__device__ __forceinline__ cx<float> rmul(float a, cx<float> u) { return up(__fmul2_rn(pk(u), bc(a))); }
__device__ __forceinline__ cx<float> rfma(float a, cx<float> u, cx<float> acc) {
    return up(__ffma2_rn(pk(u), bc(a), pk(acc)));
}
__device__ __forceinline__ cx<float> add_i(cx<float> a, cx<float> b) { return up(__fadd2_rn(pk(a), pk_i(b))); }
__device__ __forceinline__ cx<float> sub_i(cx<float> a, cx<float> b) { return up(__fadd2_rn(pk(a), pk_mi(b))); }
__device__ __forceinline__ cx<float> axmi(float k, cx<float> w, cx<float> v) {
    return up(__ffma2_rn(pk_mi(w), bc(k), pk(v)));
}

// 1/sqrt(x) for x >= 1e-36: hardware seed (MUFU.RSQ64H / MUFU.RSQ) + Newton steps, no
// special-case branches (the caller excludes zero and subnormal arguments)
__device__ __forceinline__ double rsqrt_pos(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double hx = 0.5 * x;
#pragma unroll
    for (int it = 0; it < 2; ++it) {                 // 2^-20 -> 2^-40 -> 2^-80
        const double h = fma(-hx * y, y, 0.5);       // (1 - x y^2) / 2
        y = fma(y, h, y);
    }
    return y;
}
__device__ __forceinline__ float rsqrt_approx(float x) {       // MUFU.RSQ, 2 ulp, no special cases
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rsqrt_pos(float x) {
    float y = rsqrt_approx(x);
    const float h = fmaf(-0.5f * x * y, y, 0.5f);
    return fmaf(y, h, y);
}

// Taylor coefficients of the scalar-phase sin/cos, kept in the kernel-parameter constant bank
// so that every DFMA/FFMA takes its coefficient as a constant operand (as immediates each
// fp64 coefficient costs two register moves per use).
//   cos x = 1 + z (c[0] + z (c[1] + ... + z c[6])),        c[k] = (-1)^(k+1) / (2k+2)!
//   sin x = x + x z (s[0] + z (s[1] + ... + z s[5])),      s[k] = (-1)^(k+1) / (2k+3)!,  z = x^2
struct SinCosTable {
    double c[7], s[6];
    float cf[7], sf[6];
};
__device__ __forceinline__ const double* sc_cos(const SinCosTable& t, double) { return t.c; }
__device__ __forceinline__ const double* sc_sin(const SinCosTable& t, double) { return t.s; }
__device__ __forceinline__ const float* sc_cos(const SinCosTable& t, float) { return t.cf; }
__device__ __forceinline__ const float* sc_sin(const SinCosTable& t, float) { return t.sf; }

// sin/cos of the scalar interaction phase for |x| <= 2^-4 (always the case at the
// paper's scaled amplitudes): Taylor polynomials in x^2 to x^13 / x^14, remainder
// < 2^-80, branch free so that the chain interleaves with the spin-density arithmetic.
template <typename T>
__device__ __forceinline__ void sincos_small(T x, const SinCosTable& t, T* s, T* c) {
    const T z = x * x;
    const T* cc = sc_cos(t, x);
    const T* cs = sc_sin(t, x);
    T pc = cc[6], ps = cs[5];
#pragma unroll
    for (int k = 5; k >= 0; --k) pc = fma(z, pc, cc[k]);
#pragma unroll
    for (int k = 4; k >= 0; --k) ps = fma(z, ps, cs[k]);
    *c = fma(z, pc, (T)1);
    *s = fma(x * z, ps, x);
}
// the same with cos x - 1 instead of cos x: the small quantity is kept to its own relative
// precision instead of being rounded onto 1 (see interaction(), phase modes)
template <typename T>
__device__ __forceinline__ void sincos_small_m1(T x, const SinCosTable& t, T* s, T* cm1) {
    const T z = x * x;
    const T* cc = sc_cos(t, x);
    const T* cs = sc_sin(t, x);
    T pc = cc[6], ps = cs[5];
#pragma unroll
    for (int k = 5; k >= 0; --k) pc = fma(z, pc, cc[k]);
#pragma unroll
    for (int k = 4; k >= 0; --k) ps = fma(z, ps, cs[k]);
    *cm1 = z * pc;
    *s = fma(x * z, ps, x);
}
__device__ __forceinline__ void sincos_lib(double x, double* s, double* c) { sincos(x, s, c); }
__device__ __forceinline__ void sincos_lib(float x, float* s, float* c) { sincosf(x, s, c); }

// element of the state in HBM (storage type S) <-> registers (arithmetic type T)
template <typename T, typename S>
__device__ __forceinline__ cx<T> ld_state(const typename vec2<S>::type* p) {
    const typename vec2<S>::type v = *p;
    return mk<T>((T)v.x, (T)v.y);
}
template <typename T, typename S>
__device__ __forceinline__ void st_state(typename vec2<S>::type* p, cx<T> z) {
    typename vec2<S>::type v;
    v.x = (S)z.re; v.y = (S)z.im;              // round to nearest when S is narrower than T
    *p = v;
}

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
        Fw[j] = add_i(b, a);
        Bw[j] = add_i(a, b);
    }
}

template <typename T>
__device__ __forceinline__ void kin_update(Site<T>& s, int sigma, const cx<T> Fw[5], const cx<T> Bw[5],
                                           const cx<T> Fprev[5], const cx<T> Bnext[5]) {
#pragma unroll
    for (int j = 0; j < 5; ++j) {
        s.q[j][sigma]     = sub_i(Fprev[j], Bw[j]);
        s.q[j][1 - sigma] = sub_i(Bnext[j], Fw[j]);
    }
}

// ---------------------------------------------------------------------------
// Interaction.  Constants of one application (already multiplied by the
// sub-step fraction s and by the deferred-scaling factor 4^-e):
//   g0 = s c0, g1 = s c1, g2 = s c2 / 5.
// thr[p-1] = largest angle for which a degree-p polynomial meets the tolerance.
// ---------------------------------------------------------------------------
#ifndef QLGA_FUSED_STAGES
#define QLGA_FUSED_STAGES 1      // inner Horner stages of the gauge path in one sweep (horner_stage_fused)
#endif
#ifndef QLGA_FUSED_LAST
#define QLGA_FUSED_LAST 0        // 1: the last stage (k = 1) too (five or six roundings at full magnitude instead of one)
#endif
constexpr int QLGA_PMAX = 12;
constexpr int QLGA_LUT_BASE = 83 * 16;      // theta = 2^-44: below it degree 1 serves every tolerance in use
constexpr int QLGA_LUT_N = 44 * 16;         // up to theta = 1 (theta_split <= 1/2 ends the table's use)

template <typename T> struct UConst {
    T g0, g1, g2;
    T smu;                      // s mu: chemical-potential phase of this application
    float tg1, tg2;             // 2|g1| and |g2| as floats, for the angle bound (no conversions per site)
};
template <typename T> inline UConst<T> make_uconst(double g0, double g1, double g2, double smu) {
    UConst<T> u;
    u.g0 = (T)g0; u.g1 = (T)g1; u.g2 = (T)g2; u.smu = (T)smu;
    // rounded up: the bound must not fall below the true angle
    u.tg1 = nextafterf((float)(2.0 * fabs(g1)), INFINITY);
    u.tg2 = nextafterf((float)fabs(g2), INFINITY);
    return u;
}


struct ExpTable {
    // Horner ratios of the degree-p polynomial P_p(y) = b0 (1 + r1 y (1 + r2 y (... (1 + rp y)))),
    // y = -i s K: r[p-1][k] = b_k / b_{k-1} (close to 1/k), b0[p-1] close to 1.  P_p is the
    // Chebyshev-economised Taylor polynomial of exp(y) on |y| <= thr[p-1].
    double r[QLGA_PMAX][QLGA_PMAX + 1];
    double b0[QLGA_PMAX];
    float rf[QLGA_PMAX][QLGA_PMAX + 1];   // the same rounded to fp32 (no conversions in the fp32 loops)
    float b0f[QLGA_PMAX];
    double b0m1[QLGA_PMAX];     // b0 - 1, kept to its own precision (phase modes 1, 2)
    float b0m1f[QLGA_PMAX];
    int phase_mode;             // see interaction(): 0 = phase factor as (cos, -sin), 1 = as 1 + d, 2 = 1 + d with d in fp64
    float thr[QLGA_PMAX];       // thr[p-1] = largest angle degree p serves within the tolerance
    float theta_split;          // angles above this are split into equal sub-angles
    SinCosTable sc;
    // degree by table lookup: index = (bits of theta >> 19) - QLGA_LUT_BASE, i.e. the exponent and the
    // top four mantissa bits (buckets 4-6 % wide); the entry is the degree that serves the bucket's
    // upper edge, so the choice is never below the rule "smallest p with theta <= thr[p-1]"
    unsigned char plut[QLGA_LUT_N];
};

// The site's own spin gauge.  With e = F_+/|F_+| and D = diag(e^-2, e^-1, 1, e, e^2) (rows
// m = +2..-2), K' = D^-1 K D has REAL off-diagonal elements |g1 F_+| alpha_m / 2: a spin rotation
// about z that turns F into the x-z plane.  P(K) v = D P(K') D^-1 v exactly, the rank-one part keeps
// its form with psi' = D^-1 psi (time reversal commutes with rotations), so one application of
// s K' costs 68 FP instructions instead of 88; the two diagonal rotations cost 16 per vector on
// the way in and are folded into the scalar phase on the way out.
//
__device__ __forceinline__ const double* exp_ratios(const ExpTable& t, int p, double) { return t.r[p - 1]; }
__device__ __forceinline__ const float* exp_ratios(const ExpTable& t, int p, float) { return t.rf[p - 1]; }
__device__ __forceinline__ double exp_b0(const ExpTable& t, int p, double) { return t.b0[p - 1]; }
__device__ __forceinline__ float exp_b0(const ExpTable& t, int p, float) { return t.b0f[p - 1]; }
__device__ __forceinline__ double exp_b0m1(const ExpTable& t, int p, double) { return t.b0m1[p - 1]; }
__device__ __forceinline__ float exp_b0m1(const ExpTable& t, int p, float) { return t.b0m1f[p - 1]; }

// w = (s K') u  with  s K' = g1 F'.f + g2 |chi'><chi'|,
//   (F'.f u)_m = m F_z u_m + (1/2)|F_+| (alpha_{m-1} u_{m-1} + alpha_m u_{m+1}),
//   alpha_1 = alpha_-2 = 2, alpha_0 = alpha_-1 = sqrt(6)   (f_+|m> = sqrt(6 - m(m+1))|m+1>),
//   <chi'|u> = sum_m (-1)^m psi'_{-m} u_m,   chi'_m = (-1)^m conj(psi'_{-m}).
// Inputs are pre-scaled: az = g1 F_z, az2 = 2 az, a1 = g1 |F_+|, a6 = (sqrt6/2) a1.
//
// fp32 does not use the gauge: at its degree (3) the two rotations cost what the real
// coefficients save, and they add two roundings per application (measured: 1.5-2x the
// error against the oracle).  There a1 = g1 F_+ and a6 stay complex, the lowering
// element acts as a u, the raising element as conj(a) u, and psi' = psi.
template <typename T> struct SpinGauge { static constexpr bool on = sizeof(T) == 8; };
template <typename T, bool G> struct OffDiag { using type = T; };
template <typename T> struct OffDiag<T, false> { using type = cx<T>; };

template <typename T> __device__ __forceinline__ cx<T> lower(T a, cx<T> u) { return rmul(a, u); }
template <typename T> __device__ __forceinline__ cx<T> lower(cx<T> a, cx<T> u) { return cmul(a, u); }
template <typename T> __device__ __forceinline__ cx<T> lower(T a, cx<T> u, cx<T> acc) { return rfma(a, u, acc); }
template <typename T> __device__ __forceinline__ cx<T> lower(cx<T> a, cx<T> u, cx<T> acc) { return cfma(a, u, acc); }
template <typename T> __device__ __forceinline__ cx<T> raise(T a, cx<T> u, cx<T> acc) { return rfma(a, u, acc); }
template <typename T> __device__ __forceinline__ cx<T> raise(cx<T> a, cx<T> u, cx<T> acc) { return cfma_conj(a, u, acc); }

template <typename T> __device__ __forceinline__ void scale_by(T& a, T k) { a *= k; }
template <typename T> __device__ __forceinline__ void scale_by(cx<T>& a, T k) { a = rmul(k, a); }

template <typename T, typename A>
__device__ __forceinline__ void apply_sK(const cx<T> u[5], cx<T> w[5], T az, T az2, A a1, A a6,
                                         T g2, const cx<T> psi[5]) {
    // rank-one part: t = g2 <chi'|u>
    cx<T> t = cmul(psi[4], u[0]);
    t = cfma(psi[2], u[2], t);
    t = cfma(psi[0], u[4], t);
    cx<T> t2 = cmul(psi[3], u[1]);
    t2 = cfma(psi[1], u[3], t2);
    t = rmul(g2, t - t2);
    // spin part, rows m = +2..-2 (j = 0..4), Hermitian tridiagonal (real symmetric in the gauge)
    const cx<T> r0 = raise(a1, u[1], rmul(az2, u[0]));
    const cx<T> r1 = raise(a6, u[2], lower(a1, u[0], rmul(az, u[1])));
    const cx<T> r2 = raise(a6, u[3], lower(a6, u[1]));
    const cx<T> r3 = raise(a1, u[4], lower(a6, u[2], rmul(-az, u[3])));
    const cx<T> r4 = lower(a1, u[3], rmul(-az2, u[4]));
    // add t * chi'_m,  chi'_m = (-1)^m conj(psi'_{-m})
    w[0] = cfma_conj(psi[4], t, r0);
    w[1] = cfnma_conj(psi[3], t, r1);
    w[2] = cfma_conj(psi[2], t, r2);
    w[3] = cfnma_conj(psi[1], t, r3);
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

// degree for a warp-uniform angle theta <= theta_split: five instructions instead of the 45 of the
// compare tree (which the out-of-line general path still uses)
__device__ __forceinline__ int lut_degree(const ExpTable& t, float theta) {
    int k = (int)(__float_as_uint(theta) >> 19) - QLGA_LUT_BASE;
    k = max(0, min(k, QLGA_LUT_N - 1));
    return t.plut[k];
}

// Site-local coefficients of sK' (pre-scaled, see apply_sK) in the site's spin gauge.
template <typename T> struct KCoef {
    using A = typename OffDiag<T, SpinGauge<T>::on>::type;
    T az, az2, g2;
    A a1, a6;
    cx<T> e, e2;                                   // gauge phase F_+/|F_+| and its square
    cx<T> psi[5];                                  // psi' = D^-1 psi
    T rho;
    float theta;                                   // 2|g1||F| + |g2| rho, this lane
};

// Computes the coefficients from the site and rotates the site into the spin gauge in place:
// s.q[j][sigma] <- D^-1_j s.q[j][sigma],  D^-1 = diag(e^2, e, 1, conj e, conj e^2).
template <typename T>
__device__ __forceinline__ void site_coefficients(Site<T>& s, const UConst<T>& uc, KCoef<T>& kc) {
    T n[5];
    cx<T> psi[5];
#pragma unroll
    for (int j = 0; j < 5; ++j) {
        psi[j] = s.q[j][0] + s.q[j][1];
        n[j] = fma(psi[j].re, psi[j].re, psi[j].im * psi[j].im);
    }
    kc.rho = (n[0] + n[4]) + (n[1] + n[3]) + n[2];
    const T Fz = (T)2 * (n[0] - n[4]) + (n[1] - n[3]);
    // F_+ = sum_m alpha_m conj(psi_{m+1}) psi_m = 2(conj(psi_2) psi_1 + conj(psi_-1) psi_-2)
    //                                           + sqrt6 (conj(psi_1) psi_0 + conj(psi_0) psi_-1)
    cx<T> fa = cfma_conj(psi[0], psi[1], mk<T>((T)0, (T)0));
    fa = cfma_conj(psi[3], psi[4], fa);
    cx<T> fb = cfma_conj(psi[1], psi[2], mk<T>((T)0, (T)0));
    fb = cfma_conj(psi[2], psi[3], fb);
    const T rt6 = (T)2.4494897427831780981972840747059;
    const cx<T> Fp = mk<T>(fma(rt6, fb.re, (T)2 * fa.re), fma(rt6, fb.im, (T)2 * fa.im));
    const T fp2 = fma(Fp.re, Fp.re, Fp.im * Fp.im);
    // angle bound theta = 2 |g1| |F| + |g2| rho (the exact spectral norms of the two parts);
    // |F| by the approximate reciprocal square root (2 ulp; the 2^-10 margin covers it)
    const float f2 = fmaxf((float)fma(Fz, Fz, fp2), 1e-37f);
    const float Fabs = f2 * rsqrt_approx(f2);
    kc.theta = (uc.tg1 * Fabs + uc.tg2 * (float)kc.rho) * 1.0009765625f;
    kc.g2 = uc.g2;
    kc.az = uc.g1 * Fz;
    kc.az2 = kc.az + kc.az;
    const T rt6h = (T)1.2247448713915890490986420373529;          // sqrt(6)/2
    if constexpr (SpinGauge<T>::on) {
        // gauge phase e = F_+/|F_+|; a transverse spin below 1e-18 is dropped (its term is below
        // 1e-18 |g1| |u|, far under the truncation tolerance) and the gauge is the identity
        const bool tiny = !(fp2 > (T)1e-36);
        const T rinv = rsqrt_pos(tiny ? (T)1 : fp2);
        kc.e = tiny ? mk<T>((T)1, (T)0) : mk<T>(Fp.re * rinv, Fp.im * rinv);
        kc.e2 = mk<T>(fma(kc.e.re, kc.e.re, -(kc.e.im * kc.e.im)), (T)2 * kc.e.re * kc.e.im);
        kc.a1 = tiny ? (T)0 : uc.g1 * (fp2 * rinv);
        kc.a6 = rt6h * kc.a1;
#pragma unroll
        for (int sg = 0; sg < 2; ++sg) {
            s.q[0][sg] = cmul(kc.e2, s.q[0][sg]);
            s.q[1][sg] = cmul(kc.e, s.q[1][sg]);
            s.q[3][sg] = cmul_conj(s.q[3][sg], kc.e);
            s.q[4][sg] = cmul_conj(s.q[4][sg], kc.e2);
        }
#pragma unroll
        for (int j = 0; j < 5; ++j) kc.psi[j] = s.q[j][0] + s.q[j][1];
    } else {
        kc.a1 = rmul(uc.g1, Fp);
        kc.a6 = rmul(rt6h, kc.a1);
#pragma unroll
        for (int j = 0; j < 5; ++j) kc.psi[j] = psi[j];
    }
}

// Leaves the gauge and applies the scalar phase: s.q[j][sigma] <- ph D_j u_j,
// D = diag(conj e^2, conj e, 1, e, e^2).
template <typename T>
__device__ __forceinline__ void gauge_phases(const KCoef<T>& kc, cx<T> ph, cx<T> phj[5]) {
    if constexpr (SpinGauge<T>::on) {
        phj[0] = cmul_conj(ph, kc.e2);
        phj[1] = cmul_conj(ph, kc.e);
        phj[2] = ph;
        phj[3] = cmul(ph, kc.e);
        phj[4] = cmul(ph, kc.e2);
    } else {
#pragma unroll
        for (int j = 0; j < 5; ++j) phj[j] = ph;
    }
}

// One inner Horner stage in one sweep (spin gauge, real off-diagonal coefficients):
//     out_j = v_j - i kap (sK' u)_j
// accumulated term by term onto v_j with the coefficients pre-multiplied by kap: -i c u = (c u.im, -c u.re) is one FMA pair
// per term, the rank-one amplitude is rotated once (tk = -i kap g2 <chi'|u>), and the separate update v - i kap w of the
// plain form disappears: 73 instead of 78 FP64 instructions per stage and vector.  Every term is rounded at the
// magnitude of v here (five or six roundings per component instead of one), which is harmless in an INNER stage -- its
// result is multiplied by the angle in the next one -- so the last stage (k = 1) keeps the plain form.
template <typename T>
__device__ __forceinline__ void horner_stage_fused(cx<T> u[5], const cx<T> v[5], T kap, const KCoef<T>& kc) {
    const T az = kap * kc.az, az2 = kap * kc.az2, a1 = kap * kc.a1, a6 = kap * kc.a6, g2 = kap * kc.g2;
    const cx<T>* psi = kc.psi;
    cx<T> t = cmul(psi[4], u[0]);
    t = cfma(psi[2], u[2], t);
    t = cfma(psi[0], u[4], t);
    cx<T> t2 = cmul(psi[3], u[1]);
    t2 = cfma(psi[1], u[3], t2);
    t = t - t2;
    const cx<T> tk = mk<T>(g2 * t.im, -(g2 * t.re));                 // -i kap g2 <chi'|u>
    const cx<T> r0 = axmi(a1, u[1], axmi(az2, u[0], v[0]));
    const cx<T> r1 = axmi(a6, u[2], axmi(a1, u[0], axmi(az, u[1], v[1])));
    const cx<T> r2 = axmi(a6, u[3], axmi(a6, u[1], v[2]));
    const cx<T> r3 = axmi(a1, u[4], axmi(a6, u[2], axmi(-az, u[3], v[3])));
    const cx<T> r4 = axmi(a1, u[3], axmi(-az2, u[4], v[4]));
    u[0] = cfma_conj(psi[4], tk, r0);
    u[1] = cfnma_conj(psi[3], tk, r1);
    u[2] = cfma_conj(psi[2], tk, r2);
    u[3] = cfnma_conj(psi[1], tk, r3);
    u[4] = cfma_conj(psi[0], tk, r4);
}

// Plain Horner stages k = kfirst .. 1 (u <- v - i r_k sK u) of the path without the spin gauge (fp32).  A one-stage loop
// cost the fp32 kernels 33 MOVs per 47 packed FP instructions: register-pair copies of the loop-carried (re, im) pairs
// around the back edge (ptxas).  The degrees that occur in fp32 (kfirst <= 2, i.e. p <= 3) are therefore straight-line
// code, every stage writing a fresh vector; higher degrees run two stages per trip with ping-pong vectors.
template <typename T>
__device__ __forceinline__ void horner_plain_stage(const cx<T> uin[5], cx<T> uout[5], const cx<T> v[5], const KCoef<T>& kc, T ik) {
    cx<T> w[5];
    apply_sK(uin, w, kc.az, kc.az2, kc.a1, kc.a6, kc.g2, kc.psi);
#pragma unroll
    for (int j = 0; j < 5; ++j) uout[j] = axmi(ik, w[j], v[j]);
}
template <typename T>
__device__ __forceinline__ void horner_plain_stages(cx<T> u[5], const cx<T> v[5], const KCoef<T>& kc,
                                                    const T* __restrict__ r, int kfirst) {
    cx<T> a[5], b[5];
    if (kfirst == 1) {
        horner_plain_stage<T>(u, a, v, kc, r[1]);
#pragma unroll
        for (int j = 0; j < 5; ++j) u[j] = a[j];
    } else if (kfirst == 2) {
        horner_plain_stage<T>(u, a, v, kc, r[2]);
        horner_plain_stage<T>(a, b, v, kc, r[1]);
#pragma unroll
        for (int j = 0; j < 5; ++j) u[j] = b[j];
    } else if (kfirst > 2) {
        int k = kfirst;
        if (k & 1) {
            horner_plain_stage<T>(u, a, v, kc, r[k]);
#pragma unroll
            for (int j = 0; j < 5; ++j) u[j] = a[j];
            --k;
        }
#pragma unroll 1
        for (; k >= 2; k -= 2) {
            horner_plain_stage<T>(u, a, v, kc, r[k]);
            horner_plain_stage<T>(a, u, v, kc, r[k - 1]);
        }
    }
}

// u <- P_p(-i sK') v in Horner form u_{k-1} = v + r_k (-i sK') u_k, k = p..1, u_p = v
// (stage p acts on v itself: no copy).  psi, hence K, is frozen (reading R4).
template <typename T>
__device__ __forceinline__ void horner(const cx<T> v[5], cx<T> u[5], const KCoef<T>& kc,
                                       const T* __restrict__ r, int p) {
    cx<T> w[5];
    apply_sK(v, w, kc.az, kc.az2, kc.a1, kc.a6, kc.g2, kc.psi);
    {
        const T ik = r[p];
#pragma unroll
        for (int j = 0; j < 5; ++j) u[j] = axmi(ik, w[j], v[j]);
    }
    if constexpr (SpinGauge<T>::on && QLGA_FUSED_STAGES) {
        // stages p-1 .. 2 in one sweep each; the last one in the plain form (see horner_stage_fused).  (Measured at
        // config 5: 1.525 -> 1.549 GSUP/s; the first stage fused as well, which costs a copy of v: 1.524; the last
        // one too: 1.554 for 1.3x the rounding error after 20 000 steps: not taken.)
        if (p >= 2) {
            constexpr int last_plain = QLGA_FUSED_LAST ? 0 : 1;
#pragma unroll 1
            for (int k = p - 1; k > last_plain; --k) horner_stage_fused<T>(u, v, r[k], kc);
            if (!QLGA_FUSED_LAST) {
                apply_sK(u, w, kc.az, kc.az2, kc.a1, kc.a6, kc.g2, kc.psi);
                const T ik = r[1];
#pragma unroll
                for (int j = 0; j < 5; ++j) u[j] = axmi(ik, w[j], v[j]);
            }
        }
    } else {
        horner_plain_stages<T>(u, v, kc, r, p - 1);
    }
}

// General path (never taken at the paper's amplitudes): scalar phase by the library
// sincos; angles above theta_split in nsub equal sub-angles (exact: K is frozen).
// Takes the site already in its spin gauge.  Out of line and by value so that the
// common path keeps its registers.
constexpr int QLGA_NSUB_MAX = 1 << 12;      // sub-angles of the general path: angles up to 2048 rad per application
enum { FLAG_ANGLE = 1 };                    // device error word: an interaction angle was not finite or beyond the cap

template <typename T>
__device__ __noinline__ Site<T> interaction_general(Site<T> s, KCoef<T> kc, T xph, const ExpTable& tab, float theta,
                                                    int* flag) {
    int nsub = 1;
    if (theta > tab.theta_split) {
        // a non-finite or absurd angle (bad input, a corrupted state) must not turn into a loop of 2^31
        // sub-angles: cap it, raise the context's error word, let the next synchronising call report it
        const float want = ceilf(theta / tab.theta_split);
        if (!(want <= (float)QLGA_NSUB_MAX)) {
            if (flag) atomicOr(flag, FLAG_ANGLE);
            nsub = QLGA_NSUB_MAX;
        } else {
            nsub = (int)want;
        }
    }
    if (!(fabs(xph) < (T)1e30)) {
        if (flag) atomicOr(flag, FLAG_ANGLE);
        xph = (T)0;
    }
    const T inv_nsub = (T)1 / (T)nsub;
    kc.g2 *= inv_nsub; kc.az *= inv_nsub; kc.az2 *= inv_nsub;
    scale_by(kc.a1, inv_nsub); scale_by(kc.a6, inv_nsub);
    const int p = min(QLGA_PMAX, 1 + count_below(tab.thr, theta / (float)nsub * 1.0009765625f));
    T sn, cs;
    sincos_lib(xph, &sn, &cs);
    T b0n = (T)1;
    for (int rep = 0; rep < nsub; ++rep) b0n *= exp_b0(tab, p, (T)0);
    cx<T> phj[5];
    gauge_phases<T>(kc, mk<T>(b0n * cs, -(b0n * sn)), phj);
    for (int sg = 0; sg < 2; ++sg) {
        cx<T> v[5], u[5];
        for (int j = 0; j < 5; ++j) v[j] = s.q[j][sg];
        for (int rep = 0; rep < nsub; ++rep) {
            horner<T>(v, u, kc, exp_ratios(tab, p, (T)0), p);
            for (int j = 0; j < 5; ++j) v[j] = u[j];
        }
        for (int j = 0; j < 5; ++j) s.q[j][sg] = cmul(phj[j], v[j]);
    }
    return s;
}

// Apply U^{(s)} to one site.  The site may carry a power-of-two scale 2^e; the
// caller passes constants multiplied by 4^-e, which makes the result identical
// (bit for bit, barring under/overflow) to applying U to the unscaled site.
//
// Scalar phase factor ph = b0 exp(-i x), x = s (c0 rho + mu), three formulations (tab.phase_mode):
//   0  ph = (b0 cos x, -b0 sin x), result ph * u.  cos x is rounded onto 1: a modulus error of up to half an
//      ulp that repeats at every application while the density is stationary -- in fp32 3e-8 x 8e4
//      applications = 2e-3 after 20 000 steps (measured: DESIGN.md section 8).
//   1  ph = 1 + d,  d = (b0 (cos x - 1) + (b0 - 1), -b0 sin x) with cos x - 1 and b0 - 1 kept to their own
//      relative precision; result u + d u by FMA: only the unbiased rounding of the result remains.
//   2  as 1 with rho, x and d evaluated in fp64 from the fp32 amplitudes (fp32 kernels only).
// fp64 in the spin gauge keeps formulation 0 (its phase factors are the five gauge rotations times ph).
template <typename T>
__device__ __forceinline__ void interaction(Site<T>& s, const UConst<T>& uc, const ExpTable& tab, int* flag) {
    KCoef<T> kc;
    site_coefficients<T>(s, uc, kc);               // s is in its spin gauge from here on
    // The first Horner stage of component 1 needs neither the degree nor the phase: it is
    // issued before the warp-wide reductions below so that their latency (rsqrt, REDUX,
    // vote, the branch on their result) is covered by independent FP64 instructions.
    cx<T> va[5], wa[5];
#pragma unroll
    for (int j = 0; j < 5; ++j) va[j] = s.q[j][0];
    apply_sK(va, wa, kc.az, kc.az2, kc.a1, kc.a6, kc.g2, kc.psi);
    // warp-uniform angle (one polynomial degree per warp keeps the Horner loops convergent)
    const float theta = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(kc.theta)));
    const T xph = fma(uc.g0, kc.rho, uc.smu);      // scalar phase exp(-i s (c0 rho + mu))
    const bool big_phase = !__all_sync(0xffffffffu, fabs(xph) <= (T)0.0625);
    if (big_phase || theta > tab.theta_split) {
        s = interaction_general<T>(s, kc, xph, tab, theta, flag);
        return;
    }
    const int p = lut_degree(tab, theta);
    const T pb0 = exp_b0(tab, p, (T)0);                // constant term of the polynomial (1 - O(tol))
    const bool one_plus_d = !SpinGauge<T>::on && tab.phase_mode != 0;
    cx<T> phj[5];
    cx<T> d = mk<T>((T)0, (T)0);
    if (one_plus_d) {
        if (sizeof(T) == 4 && tab.phase_mode == 2) {
            double rho64 = 0.0;
#pragma unroll
            for (int j = 0; j < 5; ++j) {
                const double pr = (double)kc.psi[j].re, pi = (double)kc.psi[j].im;
                rho64 = fma(pr, pr, fma(pi, pi, rho64));
            }
            double sn64, cm64;
            sincos_small_m1<double>(fma((double)uc.g0, rho64, (double)uc.smu), tab.sc, &sn64, &cm64);
            const double b064 = tab.b0[p - 1];
            d = mk<T>((T)fma(b064, cm64, tab.b0m1[p - 1]), (T)(-(b064 * sn64)));
        } else {
            T sn, cm1;
            sincos_small_m1<T>(xph, tab.sc, &sn, &cm1);
            d = mk<T>(fma(pb0, cm1, exp_b0m1(tab, p, (T)0)), -(pb0 * sn));
        }
    } else {
        T sn, cs;
        sincos_small<T>(xph, tab.sc, &sn, &cs);
        gauge_phases<T>(kc, mk<T>(pb0 * cs, -(pb0 * sn)), phj);
    }
    const T* r = exp_ratios(tab, p, (T)0);
    {
        cx<T> u[5];
        const T ik = r[p];
#pragma unroll
        for (int j = 0; j < 5; ++j) u[j] = axmi(ik, wa[j], va[j]);
        if constexpr (SpinGauge<T>::on && QLGA_FUSED_STAGES) {
            if (p >= 2) {
                constexpr int last_plain = QLGA_FUSED_LAST ? 0 : 1;
#pragma unroll 1
                for (int k = p - 1; k > last_plain; --k) horner_stage_fused<T>(u, va, r[k], kc);
                if (!QLGA_FUSED_LAST) {
                    apply_sK(u, wa, kc.az, kc.az2, kc.a1, kc.a6, kc.g2, kc.psi);
                    const T ikk = r[1];
#pragma unroll
                    for (int j = 0; j < 5; ++j) u[j] = axmi(ikk, wa[j], va[j]);
                }
            }
        } else {
            horner_plain_stages<T>(u, va, kc, r, p - 1);
        }
        if (one_plus_d) {
#pragma unroll
            for (int j = 0; j < 5; ++j) s.q[j][0] = cfma(d, u[j], u[j]);
        } else {
#pragma unroll
            for (int j = 0; j < 5; ++j) s.q[j][0] = cmul(phj[j], u[j]);
        }
    }
    {
        cx<T> v[5], u[5];
#pragma unroll
        for (int j = 0; j < 5; ++j) v[j] = s.q[j][1];
        horner<T>(v, u, kc, r, p);
        if (one_plus_d) {
#pragma unroll
            for (int j = 0; j < 5; ++j) s.q[j][1] = cfma(d, u[j], u[j]);
        } else {
#pragma unroll
            for (int j = 0; j < 5; ++j) s.q[j][1] = cmul(phj[j], u[j]);
        }
    }
}

}  // namespace qlga
