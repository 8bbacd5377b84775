// qlga_api.cu -- the C ABI of libqlga.so (include/qlga.h): context, sequencing of
// the fused passes into time steps, state transfers, observables, vorticity.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <new>
#include "qlga_internal.h"

using namespace qlga;

static char g_init_err[512] = "";

// defaults of the fp32 kernels (QLGA_F32), settled by the measured error growth against the fp64 path
// (DESIGN.md section 8): none of the formulations built (phase factor as 1 + d, in fp32 or fp64; tighter
// truncation; Taylor instead of economised coefficients) changes the order of magnitude of the fp32 error at
// the stated step counts, so the fastest one stays the default and QLGA_F32X is the accurate variant
#ifndef QLGA_F32_PHASE_DEFAULT
#define QLGA_F32_PHASE_DEFAULT 0
#endif
#ifndef QLGA_F32_TOL_DEFAULT
#define QLGA_F32_TOL_DEFAULT -27
#endif
#ifndef QLGA_F32_POLY_DEFAULT
#define QLGA_F32_POLY_DEFAULT 0
#endif
// fp64 arithmetic: truncation target 2^-58 for the whole error and 2^-65 for its modulus part.  Both are
// systematic (the same error at every application on a slowly varying state): the phase part adds up linearly,
// 2e5 applications (config 2) x 2^-58 = 7e-13; the modulus part feeds back through the density into the phase
// rate c0 rho and grows quadratically (measured: DESIGN.md section 8).
#ifndef QLGA_F64_TOL_DEFAULT
#define QLGA_F64_TOL_DEFAULT -58
#endif
#ifndef QLGA_F64_MOD_SHIFT_DEFAULT
#define QLGA_F64_MOD_SHIFT_DEFAULT 7
#endif
// QLGA_F32X rounds every amplitude to fp32 once per pass (6e-8): truncation targets 2^-44 / 2^-52 are far below that
// and below its accumulated effect (measured: the same 5.5e-6 after config 3's 20 000 steps for every target from
// 2^-58 down to 2^-32, at 1.25-1.5x the rate).
static const int F32X_TOL_LOG2 = -44, F32X_MOD_SHIFT = 8;
static const int F64_TOL_LOG2 = QLGA_F64_TOL_DEFAULT;
static const int F64_MOD_SHIFT = QLGA_F64_MOD_SHIFT_DEFAULT;
static const int F32_PHASE_MODE = QLGA_F32_PHASE_DEFAULT, F32_TOL_LOG2 = QLGA_F32_TOL_DEFAULT, F32_EXP_POLY = QLGA_F32_POLY_DEFAULT;

static qlga_status fail(const qlga_ctx* cc, qlga_status st, const char* fmt, const char* a = "") {
    qlga_ctx* c = const_cast<qlga_ctx*>(cc);
    char* dst = c ? c->err : g_init_err;
    snprintf(dst, 512, fmt, a);
    return st;
}
static qlga_status cuda_fail(qlga_ctx* c, const char* what, cudaError_t e) {
    char* dst = c ? c->err : g_init_err;
    snprintf(dst, 512, "%s: %s", what, cudaGetErrorString(e));
    return QLGA_ECUDA;
}
#define CU(ctx, call)                                                       \
    do {                                                                    \
        cudaError_t e_ = (call);                                            \
        if (e_ != cudaSuccess) return cuda_fail(ctx, #call, e_);            \
    } while (0)

// storage: QLGA_F32X keeps the state in fp32 (its arithmetic is fp64, in registers)
static size_t real_size(qlga_prec p) { return p == QLGA_F64 ? sizeof(double) : sizeof(float); }
static qlga_prec storage_prec(const qlga_ctx* c) { return c->prec == QLGA_F64 ? QLGA_F64 : QLGA_F32; }

// Every entry point runs on the context's own device, whatever device is current in the calling
// thread, and restores the caller's device on return.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const qlga_ctx* c) {
        if (c && cudaGetDevice(&prev) == cudaSuccess && prev != c->device)
            switched = cudaSetDevice(c->device) == cudaSuccess;
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;
};

static void band_drop_graphs(qlga_ctx* c);
static void band_release(qlga_ctx* c);

// ---------------------------------------------------------------------------
// The interaction polynomial.  exp(-i s K) v is evaluated as P_p(-i s K) v with P_p a
// degree-p polynomial with real coefficients b_j close to 1/j!.  A plain Taylor
// polynomial wastes accuracy at small |x|; Chebyshev economisation (Lanczos) of the
// degree-(p+4) Taylor polynomial on [-theta, theta] spreads the error evenly and buys
// a factor ~2^p: the remainder is  sum_{n>p} |beta_n| 2^(1-n)  with beta_n the scaled
// coefficient at the moment its degree is removed, ~ theta^(p+1) / ((p+1)! 2^p).
// With y = -i x the even part of P_p is a polynomial for cos x and the odd part for
// -i sin x, so the real polynomial A(x) = sum_j sigma_j b_j x^j, sigma_j = (-1)^(j/2),
// (Taylor: cos x + sin x) is economised; T_n has the parity of n, so parities never mix.
// ---------------------------------------------------------------------------
// *err_even (optional): the part of the bound that belongs to the even (cosine) part of the polynomial.  With
// y = -i x an eigencomponent is multiplied by A(x) - i B(x), A even, B odd, and |A - iB|^2 = 1 + 2 eps_A + 2 x eps_B:
// the even part's error is a MODULUS error, the odd part's a phase error.  A modulus error that repeats at
// every application changes the density, hence the rate c0 rho of the scalar phase: it grows like
// (c0 rho t / 2) x applications x bias (measured: DESIGN.md section 8), so it is bounded separately.
// *b0m1 (optional): b_0 - 1, accumulated on its own (at tolerances near 2^-64 it is below the resolution of
// 1 + x even in long double).
static long double economise(int p, long double theta, long double* b /*[p+1]*/, long double* err_even = nullptr,
                             long double* b0m1 = nullptr) {
    const int N = p + 4;
    long double beta[QLGA_PMAX + 8], fact = 1.0L, pw = 1.0L;
    for (int n = 0; n <= N; ++n) {
        if (n > 0) { fact *= (long double)n; pw *= theta; }
        const long double sigma = ((n / 2) % 2 == 0) ? 1.0L : -1.0L;
        beta[n] = sigma * pw / fact;                       // a_n theta^n
    }
    long double err = pw * theta / (fact * (long double)(N + 1));   // Taylor remainder of degree N
    long double ee = err;
    long double tc[QLGA_PMAX + 8][QLGA_PMAX + 8];          // T_n(t) = sum_k tc[n][k] t^k
    for (int n = 0; n <= N; ++n) for (int k = 0; k <= N; ++k) tc[n][k] = 0.0L;
    tc[0][0] = 1.0L; tc[1][1] = 1.0L;
    for (int n = 2; n <= N; ++n)
        for (int k = 0; k <= n; ++k)
            tc[n][k] = (k > 0 ? 2.0L * tc[n - 1][k - 1] : 0.0L) - tc[n - 2][k];
    long double c0 = 0.0L;                                 // beta[0] - 1, kept apart from the 1
    for (int n = N; n > p; --n) {                          // remove degree n
        const long double lam = beta[n] / tc[n][n];
        for (int k = 1; k <= n; ++k) beta[k] -= lam * tc[n][k];
        c0 -= lam * tc[n][0];
        beta[n] = 0.0L;
        err += fabsl(lam);
        if (n % 2 == 0) ee += fabsl(lam);                  // T_n has the parity of n
    }
    pw = 1.0L;
    for (int j = 0; j <= p; ++j) {
        if (j > 0) pw *= theta;
        const long double sigma = ((j / 2) % 2 == 0) ? 1.0L : -1.0L;
        b[j] = (j == 0) ? 1.0L + c0 : sigma * beta[j] / pw;
    }
    // the constant term is stored in double: a correction below half an ulp of 1 is lost
    const long double lost = fabsl(c0 - ((long double)(double)(1.0L + c0) - 1.0L));
    err += lost;
    ee += lost;
    if (err_even) *err_even = ee;
    if (b0m1) *b0m1 = c0;
    return err;
}

// thr[p-1]: largest theta for which the economised degree-p polynomial stays within
// tol = 2^tol_log2 (bisection on the monotone error bound); coefficients at that theta.
// poly = 1: the plain Taylor polynomial instead (b_k = 1/k!): its leading ratios 1, 1/2 and b0 = 1 are exact
// in binary floating point, which matters in fp32, where a ratio rounded by 3e-8 is the same relative
// error of the angle at every application.
static long double taylor(int p, long double theta, long double* b /*[p+1]*/, long double* err_even = nullptr,
                          long double* b0m1 = nullptr) {
    if (b0m1) *b0m1 = 0.0L;
    long double fact = 1.0L, pw = 1.0L;
    for (int k = 0; k <= p; ++k) {
        if (k > 0) { fact *= (long double)k; pw *= theta; }
        b[k] = 1.0L / fact;
    }
    const long double d1 = pw * theta / (fact * (long double)(p + 1)) * (1.0L + theta);   // first dropped term (degree p+1), with the tail's margin
    const long double d2 = d1 * theta / (long double)(p + 2);                            // the next one (degree p+2)
    if (err_even) *err_even = ((p + 1) % 2 == 0) ? d1 : d2;
    return d1;
}

// mod_shift: the even (modulus) part of the error is held to tol * 2^-mod_shift (0 = no separate bound).
static void build_exp_table(ExpTable& tab, int tol_log2, int poly = 0, int phase_mode = 0, int mod_shift = 0) {
    const long double tol = ldexpl(1.0L, tol_log2);
    const long double tol_mod = ldexpl(1.0L, tol_log2 - mod_shift);
    tab.phase_mode = phase_mode;
    for (int p = 1; p <= QLGA_PMAX; ++p) {
        long double b[QLGA_PMAX + 1];
        long double lo = 0.0L, hi = 4.0L;
        for (int it = 0; it < 200; ++it) {
            const long double mid = 0.5L * (lo + hi);
            long double ee = 0.0L;
            const long double et = poly ? taylor(p, mid, b, &ee) : economise(p, mid, b, &ee);
            // modulus error of an eigencomponent: eps_A cos x + eps_B sin x <= (even part) + theta (odd part)
            if (et <= tol && (mod_shift == 0 || ee + mid * et <= tol_mod)) lo = mid; else hi = mid;
        }
        long double th = lo * 0.999L;                      // margin for the fp32 angle estimate
        long double c0 = 0.0L;
        if (poly) taylor(p, th, b, nullptr, &c0); else economise(p, th, b, nullptr, &c0);
        tab.thr[p - 1] = (float)th;
        if ((long double)tab.thr[p - 1] > th) tab.thr[p - 1] = nextafterf(tab.thr[p - 1], 0.0f);
        // with a separate modulus bound a degree can serve less than the one below it: the rule "smallest p with
        // theta <= thr[p-1]" then never picks it; keep the thresholds ascending for the compare tree
        if (p > 1 && tab.thr[p - 1] < tab.thr[p - 2]) tab.thr[p - 1] = tab.thr[p - 2];
        tab.b0[p - 1] = (double)b[0];
        tab.b0m1[p - 1] = (double)c0;
        tab.b0m1f[p - 1] = (float)tab.b0m1[p - 1];
        for (int k = 0; k <= QLGA_PMAX; ++k) tab.r[p - 1][k] = 0.0;
        for (int k = 1; k <= p; ++k) tab.r[p - 1][k] = (double)(b[k] / b[k - 1]);
        tab.b0f[p - 1] = (float)tab.b0[p - 1];
        for (int k = 0; k <= QLGA_PMAX; ++k) tab.rf[p - 1][k] = (float)tab.r[p - 1][k];
    }
    const double top = tab.thr[QLGA_PMAX - 1];
    tab.theta_split = (float)(top < 0.5 ? top : 0.5);
    // degree lookup table: bucket k holds the angles whose float bits >> 19 equal QLGA_LUT_BASE + k
    for (int k = 0; k < QLGA_LUT_N; ++k) {
        const uint32_t next = (uint32_t)(QLGA_LUT_BASE + k + 1) << 19;      // first float of the next bucket
        float upper;
        memcpy(&upper, &next, sizeof(upper));
        int p = 1;
        for (int j = 0; j < QLGA_PMAX; ++j) p += (upper > tab.thr[j]) ? 1 : 0;
        tab.plut[k] = (unsigned char)(p > QLGA_PMAX ? QLGA_PMAX : p);        // theta <= theta_split <= thr[PMAX-1]
    }
    // Taylor coefficients of the scalar phase (qlga_math.cuh, sincos_small)
    long double f = 1.0L;                                  // running factorial
    for (int k = 0; k < 7; ++k) {
        f *= (long double)(2 * k + 1) * (long double)(2 * k + 2);          // (2k+2)!
        const long double sg = (k % 2 == 0) ? -1.0L : 1.0L;
        tab.sc.c[k] = (double)(sg / f);
        tab.sc.cf[k] = (float)tab.sc.c[k];
        if (k < 6) {
            tab.sc.s[k] = (double)(sg / (f * (long double)(2 * k + 3)));    // (2k+3)!
            tab.sc.sf[k] = (float)tab.sc.s[k];
        }
    }
}

// Introspection of the polynomial table (host only, no GPU): used by the CPU tests.
extern "C" qlga_status qlga_exp_polynomial(int tol_log2, int mod_shift, int p, double* theta_max, double* b0,
                                           double* r /* [p+1], r[0] unused */) {
    if (p < 1 || p > QLGA_PMAX || tol_log2 > -8 || tol_log2 < -100 || mod_shift < 0 || mod_shift > 16 || !theta_max || !b0 || !r)
        return QLGA_EINVAL;
    static ExpTable tab;                                   // 1.3 KB: keep it off the stack
    build_exp_table(tab, tol_log2, 0, 0, mod_shift);
    *theta_max = tab.thr[p - 1];
    *b0 = tab.b0[p - 1];
    for (int k = 0; k <= p; ++k) r[k] = tab.r[p - 1][k];
    return QLGA_OK;
}

// The degree the kernels' lookup table gives for a warp-uniform angle theta (host only).
extern "C" qlga_status qlga_exp_degree(int tol_log2, int mod_shift, double theta, int* p) {
    if (tol_log2 > -8 || tol_log2 < -100 || mod_shift < 0 || mod_shift > 16 || !p || !(theta >= 0.0)) return QLGA_EINVAL;
    static ExpTable tab;
    build_exp_table(tab, tol_log2, 0, 0, mod_shift);
    if (theta > tab.theta_split) return QLGA_EINVAL;          // the kernels split such angles first
    const float th = (float)theta;
    uint32_t bits;
    memcpy(&bits, &th, sizeof(bits));
    int k = (int)(bits >> 19) - QLGA_LUT_BASE;
    k = k < 0 ? 0 : (k > QLGA_LUT_N - 1 ? QLGA_LUT_N - 1 : k);
    *p = tab.plut[k];
    return QLGA_OK;
}

extern "C" const char* qlga_version(void) { return "qlga-b200 0.2 (sm_100a)"; }

// lattice extents from the caller's dims[]: {Nx, Ny} for ndim 1 and 2 (Ny = 1 in 1D),
// {Nx, Ny, Nz} for ndim 3.  Returns false on bad arguments.
static bool lattice_dims(int ndim, const int64_t* dims, int64_t& nx, int64_t& ny, int64_t& nz) {
    if (!dims || ndim < 1 || ndim > 3) return false;
    nx = dims[0]; ny = dims[1]; nz = (ndim == 3) ? dims[2] : 1;
    if (nx < 1 || ny < 1 || nz < 1 || (ndim == 1 && ny != 1)) return false;
    if ((double)nx * (double)ny * (double)nz > 1.0e12) return false;
    return true;
}

extern "C" size_t qlga_state_bytes(int ndim, const int64_t* dims, qlga_prec prec) {
    int64_t nx, ny, nz;
    if (!lattice_dims(ndim, dims, nx, ny, nz)) return 0;
    if (prec != QLGA_F64 && prec != QLGA_F32 && prec != QLGA_F32X) return 0;
    return (size_t)10 * (size_t)nx * (size_t)ny * (size_t)nz * 2 * real_size(prec);
}

extern "C" qlga_status qlga_init(qlga_ctx** out, int ndim, const int64_t* dims,
                                 double c0, double c1, double c2, qlga_order order, qlga_prec prec,
                                 void* dev_buf_a, void* dev_buf_b, void* dev_buf_c, size_t buf_bytes,
                                 void* cuda_stream) {
    if (!out) return fail(nullptr, QLGA_EINVAL, "qlga_init: out is NULL");
    *out = nullptr;
    const size_t need = qlga_state_bytes(ndim, dims, prec);
    if (need == 0) return fail(nullptr, QLGA_EINVAL, "qlga_init: bad ndim/dims/prec");
    if (order != QLGA_PLAIN && order != QLGA_INTERLEAVED)
        return fail(nullptr, QLGA_EINVAL, "qlga_init: bad order");
    if (!isfinite(c0) || !isfinite(c1) || !isfinite(c2))
        return fail(nullptr, QLGA_EINVAL, "qlga_init: non-finite coupling");
    if (!dev_buf_a || !dev_buf_b || dev_buf_a == dev_buf_b || buf_bytes < need)
        return fail(nullptr, QLGA_EINVAL, "qlga_init: need two distinct device buffers of qlga_state_bytes()");
    if (((uintptr_t)dev_buf_a | (uintptr_t)dev_buf_b | (uintptr_t)dev_buf_c) & 15)
        return fail(nullptr, QLGA_EINVAL, "qlga_init: device buffers must be 16-byte aligned");
    if (dev_buf_c && (dev_buf_c == dev_buf_a || dev_buf_c == dev_buf_b))
        return fail(nullptr, QLGA_EINVAL, "qlga_init: dev_buf_c aliases another buffer");

    // the context lives on the device that holds its buffers, whatever device is current in this thread
    int dev = -1;
    {
        void* bufs[3] = {dev_buf_a, dev_buf_b, dev_buf_c};
        for (int k = 0; k < 3; ++k) {
            if (!bufs[k]) continue;
            cudaPointerAttributes at;
            cudaError_t e = cudaPointerGetAttributes(&at, bufs[k]);
            if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail(nullptr, "qlga_init: cudaPointerGetAttributes", e); }
            if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)
                return fail(nullptr, QLGA_EINVAL, "qlga_init: the state buffers must be device memory");
            if (dev >= 0 && at.device != dev)
                return fail(nullptr, QLGA_EINVAL, "qlga_init: the state buffers live on different devices");
            dev = at.device;
        }
    }
    int caller_dev = -1;
    CU(nullptr, cudaGetDevice(&caller_dev));
    cudaDeviceProp prop;
    CU(nullptr, cudaGetDeviceProperties(&prop, dev));
    if (prop.major < 10) return fail(nullptr, QLGA_ECUDA, "qlga_init: the library is built for sm_100a only");

    qlga_ctx* c = new (std::nothrow) qlga_ctx;
    if (!c) return fail(nullptr, QLGA_ENOMEM, "qlga_init: out of host memory");
    memset(c, 0, sizeof(*c));
    c->device = dev;
    DeviceGuard guard(c);
    (void)caller_dev;
    c->ndim = ndim;
    lattice_dims(ndim, dims, c->nx, c->ny, c->nz);
    c->c[0] = c0; c->c[1] = c1; c->c[2] = c2;
    c->order = order; c->prec = prec;
    c->buf[0] = dev_buf_a; c->buf[1] = dev_buf_b; c->buf[2] = dev_buf_c;
    c->buf_bytes = buf_bytes;
    c->stream = (cudaStream_t)cuda_stream;
    c->cur = 0; c->prev = -1; c->have_state = 0; c->step = 0; c->launches = 0;
    c->path = 0; c->steps_per_launch = 0; c->threads_x = 0; c->tile_y = 0; c->fuse_plain_u = 1; c->march = 1;
    c->band = -1; c->band_rows = 0; c->band_slots = 0;
    c->tol_log2 = (prec == QLGA_F32) ? F32_TOL_LOG2 : (prec == QLGA_F32X ? F32X_TOL_LOG2 : F64_TOL_LOG2);
    c->exp_poly = (prec == QLGA_F32) ? F32_EXP_POLY : 0;
    c->f32_phase = F32_PHASE_MODE;
    c->exp_mod_shift = (prec == QLGA_F32) ? 0 : (prec == QLGA_F32X ? F32X_MOD_SHIFT : F64_MOD_SHIFT);
    build_exp_table(c->tab, c->tol_log2, c->exp_poly, c->f32_phase, c->exp_mod_shift);
    c->obs_blocks = prop.multiProcessorCount * 8;
    cudaError_t e = cudaMalloc(&c->d_partials, sizeof(double) * (size_t)c->obs_blocks * OBS_NACC);
    if (e == cudaSuccess) e = cudaMalloc(&c->d_sums, sizeof(double) * OBS_NACC);
    if (e == cudaSuccess) e = cudaMalloc(&c->d_flag, sizeof(int));
    if (e == cudaSuccess) e = cudaMemset(c->d_flag, 0, sizeof(int));
    if (e != cudaSuccess) {
        cudaFree(c->d_partials); cudaFree(c->d_sums); cudaFree(c->d_flag);
        delete c;
        return cuda_fail(nullptr, "qlga_init: cudaMalloc(scratch)", e);
    }
    c->d_stage = nullptr; c->stage_bytes = 0;
    c->err[0] = 0;
    *out = c;
    return QLGA_OK;
}

extern "C" qlga_status qlga_destroy(qlga_ctx* c) {
    if (!c) return QLGA_EINVAL;
    DeviceGuard guard(c);
    cudaStreamSynchronize(c->stream);
    cudaFree(c->d_partials); cudaFree(c->d_sums); cudaFree(c->d_stage); cudaFree(c->d_scratch); cudaFree(c->d_flag);
    band_release(c);
    if (c->prof_ev) {
        for (int k = 0; k < PROF_CAP; ++k) cudaEventDestroy(c->prof_ev[k]);
        free(c->prof_ev); free(c->prof_kind);
    }
    delete c;
    return QLGA_OK;
}

extern "C" const char* qlga_last_error(const qlga_ctx* c) { return c ? c->err : g_init_err; }
extern "C" int64_t qlga_launch_count(const qlga_ctx* c) { return c ? c->launches : -1; }

extern "C" qlga_status qlga_set_option(qlga_ctx* c, qlga_option key, int64_t v) {
    if (!c) return QLGA_EINVAL;
    {   // the instantiated band graphs hold kernel arguments (tables, tile choices): drop them on any change
        DeviceGuard guard(c);
        band_drop_graphs(c);
    }
    switch ((int)key) {
        case QLGA_OPT_PATH:
            if (v != 0 && v != 1) return fail(c, QLGA_EINVAL, "QLGA_OPT_PATH: 0 or 1");
            c->path = (int)v; return QLGA_OK;
        case QLGA_OPT_STEPS_PER_LAUNCH:
            if (v < 0 || v > max_ksteps(256) / 2) return fail(c, QLGA_EINVAL, "QLGA_OPT_STEPS_PER_LAUNCH: 0..15");
            c->steps_per_launch = (int)v; return QLGA_OK;
        case QLGA_OPT_EXP_TOL_LOG2:
            if (v > -8 || v < -100) return fail(c, QLGA_EINVAL, "QLGA_OPT_EXP_TOL_LOG2: -100..-8");
            c->tol_log2 = (int)v; build_exp_table(c->tab, c->tol_log2, c->exp_poly, c->f32_phase, c->exp_mod_shift); return QLGA_OK;
        case QLGA_OPT_THREADS_X:
            if (!pass_tile_supported(0, (int)v, 1)) return fail(c, QLGA_EINVAL, "QLGA_OPT_THREADS_X: 0, 64, 96, 128, 192, 256");
            c->threads_x = (int)v; return QLGA_OK;
        case QLGA_OPT_THREADS_Y:
            // validated as a pair with the columns per CTA: only the pairs listed in qlga.h are built
            if (v < 0 || v > 256 || !pass_tile_supported(1, (int)v, c->tile_y))
                return fail(c, QLGA_EINVAL, "QLGA_OPT_THREADS_Y: no kernel for this (TILE_Y, THREADS_Y) pair; see qlga.h");
            c->threads_y = (int)v; return QLGA_OK;
        case QLGA_OPT_TILE_Y:
            if (v < 0 || v > 8 || !pass_tile_supported(1, c->threads_y, (int)v))
                return fail(c, QLGA_EINVAL, "QLGA_OPT_TILE_Y: no kernel for this (TILE_Y, THREADS_Y) pair; see qlga.h");
            c->tile_y = (int)v; return QLGA_OK;
        case QLGA_OPT_F32_PHASE:
            if (v < 0 || v > 2) return fail(c, QLGA_EINVAL, "QLGA_OPT_F32_PHASE: 0, 1 or 2");
            c->f32_phase = (int)v; build_exp_table(c->tab, c->tol_log2, c->exp_poly, c->f32_phase, c->exp_mod_shift); return QLGA_OK;
        case QLGA_OPT_MARCH:
            if (v != 0 && v != 1) return fail(c, QLGA_EINVAL, "QLGA_OPT_MARCH: 0 or 1");
            c->march = (int)v; return QLGA_OK;
        case QLGA_OPT_EXP_MOD_SHIFT:
            if (v < 0 || v > 16) return fail(c, QLGA_EINVAL, "QLGA_OPT_EXP_MOD_SHIFT: 0..16");
            c->exp_mod_shift = (int)v; build_exp_table(c->tab, c->tol_log2, c->exp_poly, c->f32_phase, c->exp_mod_shift); return QLGA_OK;
        case QLGA_OPT_EXP_POLY:
            if (v != 0 && v != 1) return fail(c, QLGA_EINVAL, "QLGA_OPT_EXP_POLY: 0 (economised) or 1 (Taylor)");
            c->exp_poly = (int)v; build_exp_table(c->tab, c->tol_log2, c->exp_poly, c->f32_phase, c->exp_mod_shift); return QLGA_OK;
        case QLGA_OPT_FUSE_PLAIN_U:
            if (v != 0 && v != 1) return fail(c, QLGA_EINVAL, "QLGA_OPT_FUSE_PLAIN_U: 0 or 1");
            c->fuse_plain_u = (int)v; return QLGA_OK;
        case QLGA_OPT_BAND:
            if (v < -1 || v > 2) return fail(c, QLGA_EINVAL, "QLGA_OPT_BAND: -1 (auto), 0, 1 or 2");
            c->band = (int)v; return QLGA_OK;
        case QLGA_OPT_BAND_ROWS:
            if (v < 0 || v > 4096) return fail(c, QLGA_EINVAL, "QLGA_OPT_BAND_ROWS: 0 (auto) or 1..4096");
            c->band_rows = (int)v; return QLGA_OK;
        case QLGA_OPT_BAND_SLOTS:
            if (v != 0 && (v < 2 || v > 8)) return fail(c, QLGA_EINVAL, "QLGA_OPT_BAND_SLOTS: 0 (auto) or 2..8");
            c->band_slots = (int)v; return QLGA_OK;
    }
    return fail(c, QLGA_EINVAL, "qlga_set_option: unknown key");
}

// ---------------------------------------------------------------------------
// kernel timing hooks
// ---------------------------------------------------------------------------
static inline void prof_mark(qlga_ctx* c, int kind) {
    if (!c->prof_on || c->prof_n >= PROF_CAP) return;
    if (kind < 0 && (c->prof_n == 0 || c->prof_kind[c->prof_n - 1] < 0)) return;   // nothing to close
    if (cudaEventRecord(c->prof_ev[c->prof_n], c->stream) != cudaSuccess) { cudaGetLastError(); return; }
    c->prof_kind[c->prof_n++] = (signed char)kind;
}

extern "C" qlga_status qlga_profile_enable(qlga_ctx* c, int on) {
    if (!c) return QLGA_EINVAL;
    DeviceGuard guard(c);
    if (on && !c->prof_ev) {
        c->prof_ev = (cudaEvent_t*)calloc(PROF_CAP, sizeof(cudaEvent_t));
        c->prof_kind = (signed char*)calloc(PROF_CAP, 1);
        if (!c->prof_ev || !c->prof_kind) return fail(c, QLGA_ENOMEM, "qlga_profile_enable: out of host memory");
        for (int k = 0; k < PROF_CAP; ++k) CU(c, cudaEventCreate(&c->prof_ev[k]));
    }
    c->prof_on = on ? 1 : 0;
    c->prof_n = 0;
    return QLGA_OK;
}

extern "C" qlga_status qlga_profile_read(qlga_ctx* c, qlga_profile* out) {
    if (!c || !out) return c ? fail(c, QLGA_EINVAL, "qlga_profile_read: NULL") : QLGA_EINVAL;
    DeviceGuard guard(c);
    memset(out, 0, sizeof(*out));
    CU(c, cudaStreamSynchronize(c->stream));
    for (int k = 0; k + 1 < c->prof_n; ++k) {
        const int kind = c->prof_kind[k];
        if (kind < 0) continue;
        float ms = 0.f;
        CU(c, cudaEventElapsedTime(&ms, c->prof_ev[k], c->prof_ev[k + 1]));
        out->ms[kind] += ms;
        out->launches[kind] += 1;
    }
    c->prof_n = 0;
    return QLGA_OK;
}

// ---------------------------------------------------------------------------
// state transfers
// ---------------------------------------------------------------------------
static size_t state_bytes(const qlga_ctx* c) { return (size_t)10 * c->nx * c->ny * c->nz * 2 * real_size(c->prec); }
static int64_t nsites(const qlga_ctx* c) { return c->nx * c->ny * c->nz; }

static qlga_status ensure_stage(qlga_ctx* c) {
    if (c->d_stage) return QLGA_OK;
    const size_t full = state_bytes(c) / 2;                // one psi array
    size_t want = (size_t)64 << 20;
    if (want > full) want = full;
    want = (want + 255) & ~(size_t)255;
    cudaError_t e = cudaMalloc(&c->d_stage, want);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(c, QLGA_ENOMEM, "cudaMalloc(staging) failed"); }
    c->stage_bytes = want;
    return QLGA_OK;
}

// grow-only scratch for the diagnostics that return data to the host: no cudaMalloc / cudaFree
// (implicit device synchronisations) on a path meant to run every few steps
static qlga_status ensure_scratch(qlga_ctx* c, size_t bytes) {
    if (c->scratch_bytes >= bytes && c->d_scratch) return QLGA_OK;
    if (c->d_scratch) { cudaStreamSynchronize(c->stream); cudaFree(c->d_scratch); c->d_scratch = nullptr; c->scratch_bytes = 0; }
    bytes = (bytes + 255) & ~(size_t)255;
    if (cudaMalloc(&c->d_scratch, bytes) != cudaSuccess) { cudaGetLastError(); return fail(c, QLGA_ENOMEM, "cudaMalloc(diagnostics scratch) failed"); }
    c->scratch_bytes = bytes;
    return QLGA_OK;
}

// The kernels raise the device error word when an interaction angle is not finite or beyond the cap of the
// general path (a state that is not a wavefunction: Inf / NaN / absurd amplitudes).  Calls that synchronise
// anyway read it; the stream must be idle.  Reports once and clears the word.
static qlga_status check_device_flag(qlga_ctx* c, const char* who) {
    int h = 0;
    CU(c, cudaMemcpyAsync(&h, c->d_flag, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    if (h == 0) return QLGA_OK;
    CU(c, cudaMemsetAsync(c->d_flag, 0, sizeof(int), c->stream));
    return fail(c, QLGA_ESTATE, "%s: an interaction angle was not finite or beyond the supported range "
                                "(2048 rad per application): the state is not a valid wavefunction", who);
}

extern "C" qlga_status qlga_set_state_q(qlga_ctx* c, const void* q, int src_on_device) {
    if (!c || !q) return c ? fail(c, QLGA_EINVAL, "qlga_set_state_q: NULL") : QLGA_EINVAL;
    DeviceGuard guard(c);
    CU(c, cudaMemcpyAsync(c->buf[0], q, state_bytes(c),
                          src_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, c->stream));
    if (!src_on_device) CU(c, cudaStreamSynchronize(c->stream));   // host buffer may be reused on return
    c->cur = 0; c->prev = -1; c->have_state = 1; c->step = 0;
    return QLGA_OK;
}

extern "C" qlga_status qlga_get_state_q(qlga_ctx* c, void* q, int dst_on_device) {
    if (!c || !q) return c ? fail(c, QLGA_EINVAL, "qlga_get_state_q: NULL") : QLGA_EINVAL;
    DeviceGuard guard(c);
    if (!c->have_state) return fail(c, QLGA_ESTATE, "qlga_get_state_q: no state set");
    CU(c, cudaMemcpyAsync(q, c->buf[c->cur], state_bytes(c),
                          dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, c->stream));
    return check_device_flag(c, "qlga_get_state_q");
}

extern "C" qlga_status qlga_set_state_psi(qlga_ctx* c, const void* psi, int src_on_device) {
    if (!c || !psi) return c ? fail(c, QLGA_EINVAL, "qlga_set_state_psi: NULL") : QLGA_EINVAL;
    DeviceGuard guard(c);
    const int64_t n = nsites(c);
    Launch L{c->stream, &c->launches, c->device};
    if (src_on_device) {
        CU(c, launch_split_psi(L, storage_prec(c), psi, c->buf[0], n, 0, n));
    } else {
        qlga_status st = ensure_stage(c);
        if (st != QLGA_OK) return st;
        const size_t cb = 2 * real_size(c->prec);                      // bytes per complex
        const int64_t chunk = (int64_t)(c->stage_bytes / (5 * cb));
        for (int64_t off = 0; off < n; off += chunk) {
            const int64_t cnt = (n - off < chunk) ? n - off : chunk;
            for (int j = 0; j < 5; ++j)
                CU(c, cudaMemcpyAsync((char*)c->d_stage + (size_t)j * cnt * cb,
                                      (const char*)psi + ((size_t)j * n + off) * cb, (size_t)cnt * cb,
                                      cudaMemcpyHostToDevice, c->stream));
            CU(c, launch_split_psi(L, storage_prec(c), c->d_stage, c->buf[0], n, off, cnt));
        }
        CU(c, cudaStreamSynchronize(c->stream));
    }
    c->cur = 0; c->prev = -1; c->have_state = 1; c->step = 0;
    return QLGA_OK;
}

extern "C" qlga_status qlga_get_state_psi(qlga_ctx* c, void* psi, int dst_on_device) {
    if (!c || !psi) return c ? fail(c, QLGA_EINVAL, "qlga_get_state_psi: NULL") : QLGA_EINVAL;
    DeviceGuard guard(c);
    if (!c->have_state) return fail(c, QLGA_ESTATE, "qlga_get_state_psi: no state set");
    const int64_t n = nsites(c);
    Launch L{c->stream, &c->launches, c->device};
    if (dst_on_device) {
        CU(c, launch_sum_psi(L, storage_prec(c), c->buf[c->cur], psi, n, 0, n));
    } else {
        qlga_status st = ensure_stage(c);
        if (st != QLGA_OK) return st;
        const size_t cb = 2 * real_size(c->prec);
        const int64_t chunk = (int64_t)(c->stage_bytes / (5 * cb));
        for (int64_t off = 0; off < n; off += chunk) {
            const int64_t cnt = (n - off < chunk) ? n - off : chunk;
            CU(c, launch_sum_psi(L, storage_prec(c), c->buf[c->cur], c->d_stage, n, off, cnt));
            for (int j = 0; j < 5; ++j)
                CU(c, cudaMemcpyAsync((char*)psi + ((size_t)j * n + off) * cb,
                                      (const char*)c->d_stage + (size_t)j * cnt * cb, (size_t)cnt * cb,
                                      cudaMemcpyDeviceToHost, c->stream));
        }
    }
    return check_device_flag(c, "qlga_get_state_psi");
}

// ---------------------------------------------------------------------------
// time stepping
// ---------------------------------------------------------------------------
// Constants of the interaction before factor f (0..3) of a pass.  The fused pass
// defers the factor 1/2 of every kinetic factor, so before factor f the registers
// hold 2^f q and the quadratic H_int[psi] is 4^f too large: fold 4^-f in.
static void fill_pass_consts(const qlga_ctx* c, PassParams& P, double s) {
    for (int f = 0; f < 4; ++f) {
        const double sc = s * ldexp(1.0, -2 * f);
        P.g[f][0] = sc * c->c[0];
        P.g[f][1] = sc * c->c[1];
        P.g[f][2] = sc * c->c[2] / 5.0;
    }
    P.smu = s * c->mu;
    P.utail = 0;
    P.gt[0] = s * c->c[0]; P.gt[1] = s * c->c[1]; P.gt[2] = s * c->c[2] / 5.0;
    P.out_scale = 0.0625;
    P.flag = c->d_flag;
    P.tab = c->tab;
}

static int pick_other(const qlga_ctx* c, int a, int b) {   // a buffer index different from a and b
    for (int k = 0; k < 3; ++k)
        if (k != a && k != b && c->buf[k]) return k;
    return -1;
}

// ---------------------------------------------------------------------------
// Band mode: one HBM round trip per 2D time step of the plain ordering (QLGA_OPT_BAND).
//
// eq. (108) in 2D is  X Y U  (X, Y = the four kinetic factors of a direction).  With the U of step t+1 riding on
// the end of step t's x pass, a step is [Y: marching kernel, no interaction] then [X + U: tile kernel], and Y acts
// along columns only: rows [r0, r1) of Y's output depend on rows [r0 - 4, r1 + 4) of its input and on nothing
// else.  So the lattice is cut into bands of B rows; band k's y pass writes into slot k mod S of a ring of S
// bands, band k's x pass reads that slot and writes rows of the new state.  The ring (S x B rows x 10 planes:
// about 60 MB at the defaults) is rewritten every S bands and stays resident in the 126 MB L2: the state is read
// from HBM once (by the y pass) and written once (by the x pass).  The y pass of band k+1 runs beside the x pass
// of band k (FP-bound), on the library's own streams ordered by events:
//     y_k  after x_{k-S} (its slot is free again);   x_k  after y_k;   x_k and x_{k+1} on alternating streams so
//     that one fills the SMs the other's last wave leaves idle.
// The schedule of one step is captured once into a CUDA graph per (source, destination, trailing U) and replayed.
// The kernels and their arithmetic are the two-launch path's: the results are bit-identical.
// ---------------------------------------------------------------------------
#ifdef QLGA_TRACE
static __device__ unsigned long long g_trace[2 * 8192];
extern "C" int qlga_debug_trace(unsigned long long* host_out, int reset) {
    if (reset) {
        static unsigned long long init[2 * 8192];
        for (int k = 0; k < 8192; ++k) { init[2 * k] = ~0ull; init[2 * k + 1] = 0; }
        return (int)cudaMemcpyToSymbol(g_trace, init, sizeof(init));
    }
    cudaDeviceSynchronize();
    return (int)cudaMemcpyFromSymbol(host_out, g_trace, sizeof(g_trace));
}
#endif
static int64_t band_rows_eff(const qlga_ctx* c) {
    if (c->band_rows > 0) return c->band_rows;
    const int64_t row_bytes = c->nx * 10 * 2 * (int64_t)real_size(c->prec);
    int64_t b = ((int64_t)20 << 20) / row_bytes;
    b -= b % 8;
    if (b < 8) b = 8;
    if (b > 256) b = 256;
    return b;
}
static int band_slots_eff(const qlga_ctx* c) { return c->band_slots > 0 ? c->band_slots : 3; }

static bool band_applies(const qlga_ctx* c) {
    if (c->band == 0 || c->ndim != 2 || c->order != QLGA_PLAIN || c->path != 0) return false;
    if (!c->march || c->tile_y != 0 || c->threads_y != 0 || !c->fuse_plain_u) return false;
    const int64_t B = band_rows_eff(c);
    if (c->ny < 4 * B) return false;
    if (c->band < 0) {
        // auto: only where a band's x kernel still fills the GPU (two waves of 128-thread CTAs at three per SM on 148
        // SMs; a narrow lattice would run 512 small kernels below their occupancy) and the state does not fit in L2 anyway
        const int threads = c->threads_x ? c->threads_x : 128;
        const int64_t tiles = (c->nx + threads - 9) / (threads - 8);
        if (B * tiles < 888) return false;
        if ((size_t)c->nx * c->ny * 10 * 2 * real_size(c->prec) < ((size_t)256 << 20)) return false;
    }
    return true;
}

static void band_drop_graphs(qlga_ctx* c) {
    if (c->band_ngraph > 0) cudaStreamSynchronize(c->stream);        // a replay may still be running on the caller's stream
    for (int k = 0; k < c->band_ngraph; ++k) cudaGraphExecDestroy(c->band_graph[k].exec);
    c->band_ngraph = 0;
}

static void band_release(qlga_ctx* c) {
    band_drop_graphs(c);
    for (int k = 0; k < 4; ++k) if (c->band_stream[k]) { cudaStreamDestroy(c->band_stream[k]); c->band_stream[k] = nullptr; }
    if (c->band_ev) {
        for (int k = 0; k < c->band_nev; ++k) cudaEventDestroy(c->band_ev[k]);
        free(c->band_ev); c->band_ev = nullptr; c->band_nev = 0;
    }
    if (c->d_band) cudaCtxResetPersistingL2Cache();        // the ring's lines go back to normal before its memory is reused
    cudaFree(c->d_band); c->d_band = nullptr; c->band_bytes = 0;
}

static qlga_status band_setup(qlga_ctx* c, int64_t B, int S, int64_t nb) {
    if (!c->band_stream[0]) {
        int lo = 0, hi = 0;
        CU(c, cudaDeviceGetStreamPriorityRange(&lo, &hi));
        // the y pass is short and feeds the x pass: highest priority, so that its CTAs take the first free slots
        CU(c, cudaStreamCreateWithPriority(&c->band_stream[0], cudaStreamNonBlocking, lo));
        CU(c, cudaStreamCreateWithPriority(&c->band_stream[1], cudaStreamNonBlocking, hi));
        CU(c, cudaStreamCreateWithPriority(&c->band_stream[2], cudaStreamNonBlocking, lo));
        CU(c, cudaStreamCreateWithPriority(&c->band_stream[3], cudaStreamNonBlocking, lo));
    }
    const size_t need = (size_t)S * 10 * B * c->nx * 2 * real_size(c->prec);
    if (c->band_bytes < need) {
        CU(c, cudaStreamSynchronize(c->stream));
        band_drop_graphs(c);
        cudaFree(c->d_band); c->d_band = nullptr; c->band_bytes = 0;
        if (cudaMalloc(&c->d_band, need) != cudaSuccess) { cudaGetLastError(); return fail(c, QLGA_ENOMEM, "cudaMalloc(band ring) failed"); }
        c->band_bytes = need;
        // The ring must STAY in L2: without this the dirty lines of the y pass are written back to DRAM within
        // microseconds (measured: 21.4 GB of DRAM writes per step instead of 10.7) although the x pass reads them
        // from L2.  The accesses of the library's own streams to the ring are marked persisting (the kernel nodes of
        // the captured graphs inherit the window); the device's persisting set-aside is raised to the ring's size
        // (a per-device limit: it stays raised; qlga.h).
        cudaDeviceProp prop;
        CU(c, cudaGetDeviceProperties(&prop, c->device));
        if (prop.persistingL2CacheMaxSize > 0) {
            size_t cur = 0;
            CU(c, cudaDeviceGetLimit(&cur, cudaLimitPersistingL2CacheSize));
            const size_t want = need < (size_t)prop.persistingL2CacheMaxSize ? need : (size_t)prop.persistingL2CacheMaxSize;
            if (cur < want) CU(c, cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, want));
            cudaStreamAttrValue av;
            memset(&av, 0, sizeof(av));
            av.accessPolicyWindow.base_ptr = c->d_band;
            av.accessPolicyWindow.num_bytes = need < (size_t)prop.accessPolicyMaxWindowSize ? need : (size_t)prop.accessPolicyMaxWindowSize;
            av.accessPolicyWindow.hitRatio = 1.0f;
            av.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
            av.accessPolicyWindow.missProp = cudaAccessPropertyStreaming;
            for (int k = 0; k < 4; ++k)
                CU(c, cudaStreamSetAttribute(c->band_stream[k], cudaStreamAttributeAccessPolicyWindow, &av));
        }
    }
    const int nev = (int)(2 * nb + 1);
    if (c->band_nev < nev) {
        cudaEvent_t* ev = (cudaEvent_t*)realloc(c->band_ev, sizeof(cudaEvent_t) * nev);
        if (!ev) return fail(c, QLGA_ENOMEM, "band events: out of host memory");
        c->band_ev = ev;
        for (; c->band_nev < nev; ++c->band_nev)
            CU(c, cudaEventCreateWithFlags(&c->band_ev[c->band_nev], cudaEventDisableTiming));
    }
    return QLGA_OK;
}

// issue the band schedule of one time step; `origin` is the stream the step is ordered on (the caller's stream,
// or the capture origin)
static qlga_status band_issue(qlga_ctx* c, cudaStream_t origin, int src, int dst, bool tail, int64_t B, int S) {
    const int64_t nb = (c->ny + B - 1) / B;
    cudaEvent_t* evY = c->band_ev;
    cudaEvent_t* evX = c->band_ev + nb;
    cudaEvent_t ev0 = c->band_ev[2 * nb];
    cudaStream_t sy = c->band_stream[1];
    cudaStream_t sx[2] = {c->band_stream[2], c->band_stream[3]};
    const size_t cb = 2 * real_size(c->prec);
    const int64_t slot_plane = B * c->nx;                            // elements per plane of a ring slot

    CU(c, cudaEventRecord(ev0, origin));
    CU(c, cudaStreamWaitEvent(sy, ev0, 0));
    CU(c, cudaStreamWaitEvent(sx[0], ev0, 0));
    CU(c, cudaStreamWaitEvent(sx[1], ev0, 0));

    PassParams Py, Px;
    Py.nx = c->nx; Py.ny = c->ny; Py.nz = 1;
    fill_pass_consts(c, Py, 1.0);
    Py.ksteps = 1; Py.umode = 0; Py.utail = 0;
    Px = Py;
    Px.utail = tail ? 1 : 0;
    Py.src = c->buf[src];
    Py.dst_plane = slot_plane;
    Px.src_plane = slot_plane;
    Px.dst_plane = c->nx * c->ny;

    auto issue_y = [&](int64_t k) -> qlga_status {
        if (k >= S) CU(c, cudaStreamWaitEvent(sy, evX[k - S], 0));
        Launch L{sy, &c->launches, c->device};
        Py.dst = (char*)c->d_band + (size_t)(k % S) * 10 * slot_plane * cb;
        Py.row_begin = k * B;
        Py.row_end = (k + 1) * B < c->ny ? (k + 1) * B : c->ny;
        Py.dst_row_origin = k * B;
#ifdef QLGA_TRACE
        { void* tp = nullptr; cudaGetSymbolAddress(&tp, g_trace); Py.trace = (unsigned long long*)tp; Py.trace_id = (int)(2 * k) + 2048 * (c->band_ngraph & 3); }   // debug build: graph n traces into ids [2048 n, 2048 n + 2 bands)
#endif
        CU(c, launch_march(L, c->prec, 1, Py));
        CU(c, cudaEventRecord(evY[k], sy));
        return QLGA_OK;
    };
    auto issue_x = [&](int64_t k) -> qlga_status {
        cudaStream_t s = sx[k & 1];
        CU(c, cudaStreamWaitEvent(s, evY[k], 0));
        Launch L{s, &c->launches, c->device};
        const int64_t r0 = k * B, r1 = (k + 1) * B < c->ny ? (k + 1) * B : c->ny;
        Px.ny = r1 - r0;
        Px.src = (const char*)c->d_band + (size_t)(k % S) * 10 * slot_plane * cb;
        Px.dst = (char*)c->buf[dst] + (size_t)r0 * c->nx * cb;
#ifdef QLGA_TRACE
        { void* tp = nullptr; cudaGetSymbolAddress(&tp, g_trace); Px.trace = (unsigned long long*)tp; Px.trace_id = (int)(2 * k + 1) + 2048 * (c->band_ngraph & 3); }
#endif
        CU(c, launch_pass(L, c->prec, 0, Px, c->threads_x, 1));
        CU(c, cudaEventRecord(evX[k], s));
        return QLGA_OK;
    };
    qlga_status st;
    for (int64_t k = 0; k < S && k < nb; ++k)
        if ((st = issue_y(k)) != QLGA_OK) return st;
    for (int64_t k = 0; k < nb; ++k) {
        if ((st = issue_x(k)) != QLGA_OK) return st;
        if (k + S < nb && (st = issue_y(k + S)) != QLGA_OK) return st;
    }
    // join: each x stream is ordered, so its last event covers it; every y precedes an x
    CU(c, cudaStreamWaitEvent(origin, evX[nb - 1], 0));
    if (nb >= 2) CU(c, cudaStreamWaitEvent(origin, evX[nb - 2], 0));
    return QLGA_OK;
}

static qlga_status step_band(qlga_ctx* c, int src, int dst, bool tail) {
    const int64_t B = band_rows_eff(c);
    const int S = band_slots_eff(c);
    const int64_t nb = (c->ny + B - 1) / B;
    qlga_status st = band_setup(c, B, S, nb);
    if (st != QLGA_OK) return st;
    if (c->band == 1) return band_issue(c, c->stream, src, dst, tail, B, S);      // -1 (auto) and 2: the graph

    qlga_ctx::BandGraph* g = nullptr;
    for (int k = 0; k < c->band_ngraph; ++k) {
        qlga_ctx::BandGraph& h = c->band_graph[k];
        if (h.src == src && h.dst == dst && h.tail == (int)tail && h.rows == B && h.slots == S) { g = &h; break; }
    }
    if (!g) {
        if (c->band_ngraph == 12) band_drop_graphs(c);
        // (the per-device shared-memory opt-in of the x pass, run_pass, was made by the first step of the call,
        // which always takes the two-launch path: nothing but launches, event records and waits is captured)
        const int64_t before = c->launches;
        cudaGraph_t graph = nullptr;
        CU(c, cudaStreamBeginCapture(c->band_stream[0], cudaStreamCaptureModeRelaxed));
        st = band_issue(c, c->band_stream[0], src, dst, tail, B, S);
        cudaError_t e = cudaStreamEndCapture(c->band_stream[0], &graph);
        const int64_t nodes = c->launches - before;
        c->launches = before;
        if (st != QLGA_OK) { if (graph) cudaGraphDestroy(graph); cudaGetLastError(); return st; }
        if (e != cudaSuccess) return cuda_fail(c, "cudaStreamEndCapture(band schedule)", e);
        cudaGraphExec_t exec = nullptr;
        e = cudaGraphInstantiate(&exec, graph, 0);
        cudaGraphDestroy(graph);
        if (e != cudaSuccess) return cuda_fail(c, "cudaGraphInstantiate(band schedule)", e);
        g = &c->band_graph[c->band_ngraph++];
        g->src = src; g->dst = dst; g->tail = (int)tail; g->rows = B; g->slots = S; g->exec = exec; g->nodes = nodes;
    }
    CU(c, cudaGraphLaunch(g->exec, c->stream));
    c->launches += g->nodes;
    return QLGA_OK;
}

static qlga_status step_fused(qlga_ctx* c, int64_t nsteps) {
    Launch L{c->stream, &c->launches, c->device};
    const bool inter = c->order == QLGA_INTERLEAVED;
    const double s = inter ? 1.0 / (4.0 * c->ndim) : 1.0;
    PassParams P;
    P.nx = c->nx; P.ny = c->ny; P.nz = c->nz;
    fill_pass_consts(c, P, s);
    if (c->ndim == 1) {
        const int threads = c->threads_x ? c->threads_x : 128;
        int kmax = c->steps_per_launch;
        if (kmax == 0) {
            // auto: four steps per launch when the lattice is too small to fill the GPU (launch latency);
            // on a large lattice two where a step is light enough for its memory phase to count (plain
            // ordering: 2^22 sites fp64 10.5 -> 11.2, fp32 20.2 -> 23.7 GSUP/s; interleaved fp32 +3 %), one
            // for the FP64-bound interleaved step (the doubled halo recompute costs more than it saves)
            kmax = (c->nx <= 262144) ? 4 : ((!inter || c->prec == QLGA_F32) ? 2 : 1);
        }
        if (kmax > max_ksteps(threads) / 2) kmax = max_ksteps(threads) / 2;
        if (kmax < 1) kmax = 1;
        int64_t left = nsteps;
        while (left > 0) {
            // keep the very last step a single-step launch so that the previous state
            // survives in the other buffer for eq. (85)
            int k = (int)((left - 1 < kmax) ? left - 1 : kmax);
            if (k < 1) k = 1;
            const int dst = pick_other(c, c->cur, -1);
            P.src = c->buf[c->cur]; P.dst = c->buf[dst];
            P.ksteps = k; P.umode = inter ? 2 : 1;
            prof_mark(c, 0);
            CU(c, launch_pass(L, c->prec, 0, P, threads, 1));
            c->prev = (k == 1) ? c->cur : -1;
            c->cur = dst;
            left -= k; c->step += k;
        }
        return QLGA_OK;
    }
    // 2D: y pass then x pass; 3D: z, y, x (R7).  The passes ping-pong between buffers; with a
    // third buffer the state before the step survives (for eq. 85), otherwise it is overwritten.
    // Plain ordering: inside one call the U of step t+1 rides on the end of step t's x pass (see
    // pass_kernel); the first step of a call applies its own U on its first pass, the last step leaves the
    // state without a trailing U.  With a third buffer the state before the last step must be a true state
    // of the time series (eq. 85), so the last-but-one step does not carry the last step's U either.
    bool u_done = false;                                   // the coming step's U has already been applied
    const bool keeps_prev = pick_other(c, c->cur, pick_other(c, c->cur, -1)) >= 0;
    for (int64_t t = 0; t < nsteps; ++t) {
        const int start = c->cur;
        const int third = pick_other(c, start, pick_other(c, start, -1));
        int src = start;
        const bool tail = !inter && c->fuse_plain_u && (t + 1 < nsteps) && !(keeps_prev && t + 2 == nsteps);
        if (u_done && band_applies(c)) {
            // one HBM round trip: the y pass and the x pass of the step pipelined band by band through L2
            const int dst = pick_other(c, start, -1);
            prof_mark(c, 3);
            const qlga_status st = step_band(c, start, dst, tail);
            if (st != QLGA_OK) return st;
            u_done = tail;
            c->prev = (third >= 0) ? start : -1;
            c->cur = dst;
            ++c->step;
            continue;
        }
        for (int d = c->ndim - 1; d >= 0; --d) {
            int dst;
            if (third >= 0) {
                // rotate through the two buffers that do not hold the step's initial state
                const int a = pick_other(c, start, -1), b = third;
                dst = (src == a) ? b : a;
            } else {
                dst = pick_other(c, src, -1);
            }
            P.ksteps = 1;
            P.src = c->buf[src]; P.dst = c->buf[dst];
            // U is the rightmost operator of the plain step: it rides on the first pass
            P.umode = inter ? 2 : ((d == c->ndim - 1 && !u_done) ? 1 : 0);
            P.utail = (d == 0 && tail) ? 1 : 0;
            prof_mark(c, d == 0 ? 0 : 1);
            // strided passes, measured defaults.  Interleaved (FP-pipe bound): the kernel's own (fp64 one
            // column x 128 rows, fp32 two x 64); 3D fp64: two columns, i.e. whole 32-byte sectors, which the
            // page-crossing z lines need (+12 % at 512^3).  Plain ordering: the memory phases count.  A pass
            // that carries the step's U: fp64 two columns x 64 rows (8192^2: 8.8 ms against 12.2 for one
            // column), fp32 four x 64; a U-free pass (pure streaming): fp64 four x 64 (6.2 ms against 8.7 for
            // two columns), fp32 eight x 32 (3.2 against 5.3 ms)
            int cxw = c->tile_y, thr = c->threads_y;
            if (d > 0 && cxw == 0) {
                if (!inter) {
                    const bool f64 = c->prec == QLGA_F64;
                    cxw = (P.umode != 0) ? (f64 ? 2 : 4) : (f64 ? 4 : 8);
                    if (thr == 0) thr = (P.umode != 0 && f64) ? 128 : 256;
                } else if (c->ndim == 3 && c->prec == QLGA_F64) { cxw = 2; if (thr == 0) thr = 128; }
            }
            if (d > 0 && c->march && c->tile_y == 0 && c->threads_y == 0 && march_supported(d, P)) {
                // a strided pass without interaction: one thread per (column, m) marching along the line
                CU(c, launch_march(L, c->prec, d, P));
                src = dst;
                continue;
            }
            if (!pass_tile_supported(d == 0 ? 0 : 1, d == 0 ? c->threads_x : thr, d == 0 ? 1 : cxw))
                return fail(c, QLGA_EINVAL, "qlga_step: no kernel for the (TILE_Y, THREADS_Y) pair this pass resolves to; "
                                            "set both options or neither (qlga.h)");
            CU(c, launch_pass(L, c->prec, d, P, d == 0 ? c->threads_x : thr, d == 0 ? 1 : cxw));
            src = dst;
        }
        u_done = tail;
        c->prev = (third >= 0) ? start : -1;
        c->cur = src;
        ++c->step;
    }
    return QLGA_OK;
}

static qlga_status step_per_operator(qlga_ctx* c, int64_t nsteps) {
    Launch L{c->stream, &c->launches, c->device};
    const bool inter = c->order == QLGA_INTERLEAVED;
    const double s = inter ? 1.0 / (4.0 * c->ndim) : 1.0;
    const double g[3] = {s * c->c[0], s * c->c[1], s * c->c[2] / 5.0};
    for (int64_t t = 0; t < nsteps; ++t) {
        prof_mark(c, 2);
        if (!inter) CU(c, launch_interaction(L, c->prec, c->buf[c->cur], nsites(c), g, s * c->mu, c->tab, c->d_flag));
        for (int d = c->ndim - 1; d >= 0; --d)
            for (int k = 0; k < 4; ++k) {
                const int sigma = (k < 2) ? 1 : 0;                     // components 2, 2, 1, 1
                if (inter) CU(c, launch_interaction(L, c->prec, c->buf[c->cur], nsites(c), g, s * c->mu, c->tab, c->d_flag));
                const int dst = pick_other(c, c->cur, -1);
                CU(c, launch_kinetic(L, c->prec, c->buf[c->cur], c->buf[dst], c->nx, c->ny, c->nz, d, sigma));
                c->cur = dst;
            }
        c->prev = -1;
        ++c->step;
    }
    return QLGA_OK;
}

extern "C" qlga_status qlga_set_chemical_potential(qlga_ctx* c, double mu) {
    if (!c) return QLGA_EINVAL;
    if (!(mu == mu) || mu - mu != 0.0) return fail(c, QLGA_EINVAL, "qlga_set_chemical_potential: not a finite value");
    { DeviceGuard guard(c); band_drop_graphs(c); }
    c->mu = mu;
    return QLGA_OK;
}

extern "C" qlga_status qlga_step(qlga_ctx* c, int64_t n) {
    if (!c) return QLGA_EINVAL;
    DeviceGuard guard(c);
    if (n < 0) return fail(c, QLGA_EINVAL, "qlga_step: n < 0");
    if (!c->have_state) return fail(c, QLGA_ESTATE, "qlga_step: no state set");
    if (n == 0) return QLGA_OK;
    const qlga_status st = c->path == 0 ? step_fused(c, n) : step_per_operator(c, n);
    prof_mark(c, -1);
    return st;
}

// ---------------------------------------------------------------------------
// diagnostics
// ---------------------------------------------------------------------------
// extent of the slowest axis (the one a slab decomposition cuts) and sites per layer of it
static int64_t slow_extent(const qlga_ctx* c) { return c->ndim == 1 ? c->nx : (c->ndim == 2 ? c->ny : c->nz); }
static int64_t layer_sites(const qlga_ctx* c) { return nsites(c) / slow_extent(c); }

extern "C" qlga_status qlga_observable_sums(qlga_ctx* c, double* host_sums) {
    if (!c || !host_sums) return c ? fail(c, QLGA_EINVAL, "qlga_observable_sums: NULL") : QLGA_EINVAL;
    DeviceGuard guard(c);
    if (!c->have_state) return fail(c, QLGA_ESTATE, "qlga_observable_sums: no state set");
    Launch L{c->stream, &c->launches, c->device};
    const void* prev = (c->prev >= 0) ? c->buf[c->prev] : nullptr;
    const int64_t r0 = c->ghost * layer_sites(c), r1 = nsites(c) - r0;      // owned layers
    int blocks = c->obs_blocks;
    CU(c, launch_observables(L, storage_prec(c), c->buf[c->cur], prev, c->nx, c->ny, c->nz, c->ndim, r0, r1,
                             c->d_partials, blocks, c->d_sums));
    double h[OBS_NACC];
    CU(c, cudaMemcpyAsync(h, c->d_sums, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    const qlga_status fst = check_device_flag(c, "qlga_observables");       // synchronises the stream
    if (fst != QLGA_OK) return fst;
    for (int k = 0; k < 15; ++k) host_sums[k] = h[k];
    host_sums[15] = prev ? h[15] : NAN;
    host_sums[16] = prev ? h[16] : NAN;
    return QLGA_OK;
}

extern "C" qlga_status qlga_observables_from_sums(const qlga_ctx* c, const double* h, qlga_obs* out) {
    if (!c || !h || !out) return QLGA_EINVAL;
    double npsi = 0.0;
    for (int j = 0; j < 5; ++j) { out->n_m[j] = h[j]; npsi += h[j]; }
    out->norm_psi = npsi; out->norm_q = h[5];
    out->F[0] = h[6]; out->F[1] = h[7]; out->F[2] = h[8];
    out->A00_re = h[9]; out->A00_im = h[10]; out->A00_abs2 = h[11];
    out->e_kin = h[12];
    out->e_c0 = 0.5 * c->c[0] * h[13];
    out->e_c1 = 0.5 * c->c[1] * h[14];
    out->e_c2 = 0.5 * c->c[2] * h[11];
    out->e_total = out->e_kin + out->e_c0 + out->e_c1 + out->e_c2;
    // eq. (85): i (N - O)/N with O = <psi|psi_prev>:  re = Im(O)/N, im = (N - Re(O))/N
    out->e_dt_re = h[16] / npsi;                     // NaN without a previous state
    out->e_dt_im = (npsi - h[15]) / npsi;
    out->step = c->step;
    return QLGA_OK;
}

extern "C" qlga_status qlga_observables(qlga_ctx* c, qlga_obs* out) {
    if (!c || !out) return c ? fail(c, QLGA_EINVAL, "qlga_observables: NULL") : QLGA_EINVAL;
    double h[QLGA_NSUMS];
    const qlga_status st = qlga_observable_sums(c, h);
    if (st != QLGA_OK) return st;
    return qlga_observables_from_sums(c, h, out);
}

extern "C" qlga_status qlga_angle_stats(qlga_ctx* c, qlga_angles* out) {
    if (!c || !out) return c ? fail(c, QLGA_EINVAL, "qlga_angle_stats: NULL") : QLGA_EINVAL;
    DeviceGuard guard(c);
    if (!c->have_state) return fail(c, QLGA_ESTATE, "qlga_angle_stats: no state set");
    const qlga_status st = ensure_scratch(c, 15 * sizeof(unsigned long long));
    if (st != QLGA_OK) return st;
    Launch L{c->stream, &c->launches, c->device};
    const double s = c->order == QLGA_INTERLEAVED ? 1.0 / (4.0 * c->ndim) : 1.0;
    unsigned long long* d = (unsigned long long*)c->d_scratch;
    unsigned long long h[15];
    CU(c, cudaMemsetAsync(d, 0, sizeof(h), c->stream));
    int blocks = c->obs_blocks;
    if ((int64_t)blocks * 256 > nsites(c)) blocks = (int)((nsites(c) + 255) / 256);
    CU(c, launch_angle_stats(L, storage_prec(c), c->buf[c->cur], nsites(c), 2.0 * fabs(s * c->c[1]), fabs(s * c->c[2]) / 5.0,
                             s * c->c[0], s * c->mu, c->tab, blocks, d));
    CU(c, cudaMemcpyAsync(h, d, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    double sum; unsigned int mx[2];
    memcpy(&sum, &h[0], sizeof(double)); memcpy(mx, &h[1], sizeof(mx));
    float tmax, pmax;
    memcpy(&tmax, &mx[0], 4); memcpy(&pmax, &mx[1], 4);
    out->theta_max = tmax; out->theta_mean = sum / (double)nsites(c); out->phase_max = pmax;
    for (int p = 0; p < 13; ++p) out->degree_hist[p] = (int64_t)h[2 + p];
    return QLGA_OK;
}

// ---- slab decomposition: ghost / edge layers of the slowest axis ------------------------------
extern "C" qlga_status qlga_slab_configure(qlga_ctx* c, int64_t ghost) {
    if (!c) return QLGA_EINVAL;
    if (ghost < 0 || 3 * ghost > slow_extent(c))
        return fail(c, QLGA_EINVAL, "qlga_slab_configure: need 0 <= 3 * ghost <= extent of the slowest axis");
    c->ghost = ghost;
    return QLGA_OK;
}

// copies `ghost` consecutive layers starting at layer `first` of all 10 planes between the
// current state and a packed [10][ghost][layer] buffer: one strided copy (10 rows of
// ghost * layer contiguous elements, pitch = one plane)
static qlga_status slab_copy(qlga_ctx* c, const char* what, int64_t first, void* packed, bool to_packed) {
    const size_t elem = 2 * real_size(c->prec);
    const size_t width = (size_t)c->ghost * layer_sites(c) * elem;
    const size_t pitch = (size_t)nsites(c) * elem;
    char* st = (char*)c->buf[c->cur] + (size_t)first * layer_sites(c) * elem;
    cudaError_t e = to_packed
        ? cudaMemcpy2DAsync(packed, width, st, pitch, width, 10, cudaMemcpyDeviceToDevice, c->stream)
        : cudaMemcpy2DAsync(st, pitch, packed, width, width, 10, cudaMemcpyDeviceToDevice, c->stream);
    if (e != cudaSuccess) return cuda_fail(c, what, e);
    return QLGA_OK;
}

extern "C" qlga_status qlga_slab_edge_get(qlga_ctx* c, int side, void* dev_out) {
    if (!c || !dev_out || (side != 0 && side != 1))
        return c ? fail(c, QLGA_EINVAL, "qlga_slab_edge_get: bad arguments") : QLGA_EINVAL;
    DeviceGuard guard(c);
    if (!c->have_state || c->ghost <= 0) return fail(c, QLGA_ESTATE, "qlga_slab_edge_get: no state, or not a slab");
    const int64_t first = side == 0 ? c->ghost : slow_extent(c) - 2 * c->ghost;
    return slab_copy(c, "qlga_slab_edge_get", first, dev_out, true);
}

extern "C" qlga_status qlga_slab_ghost_set(qlga_ctx* c, int side, const void* dev_in) {
    if (!c || !dev_in || (side != 0 && side != 1))
        return c ? fail(c, QLGA_EINVAL, "qlga_slab_ghost_set: bad arguments") : QLGA_EINVAL;
    DeviceGuard guard(c);
    if (!c->have_state || c->ghost <= 0) return fail(c, QLGA_ESTATE, "qlga_slab_ghost_set: no state, or not a slab");
    const int64_t first = side == 0 ? 0 : slow_extent(c) - c->ghost;
    return slab_copy(c, "qlga_slab_ghost_set", first, const_cast<void*>(dev_in), false);
}

extern "C" qlga_status qlga_vorticity(qlga_ctx* c, void* omega, int dst_on_device) {
    if (!c || !omega) return c ? fail(c, QLGA_EINVAL, "qlga_vorticity: NULL") : QLGA_EINVAL;
    DeviceGuard guard(c);
    if (c->ndim != 2) return fail(c, QLGA_EUNSUP, "qlga_vorticity: 2D lattices only");
    if (!c->have_state) return fail(c, QLGA_ESTATE, "qlga_vorticity: no state set");
    Launch L{c->stream, &c->launches, c->device};
    const size_t bytes = (size_t)5 * c->nx * c->ny * real_size(c->prec);
    if (dst_on_device) {
        CU(c, launch_vorticity(L, storage_prec(c), c->buf[c->cur], omega, c->nx, c->ny));
        return QLGA_OK;
    }
    // host destination: a buffer that holds neither the current nor the previous
    // state serves as scratch (omega is a quarter of a state); else allocate
    int scratch = -1;
    for (int k = 0; k < 3; ++k)
        if (c->buf[k] && k != c->cur && k != c->prev) scratch = k;
    void* tmp = scratch >= 0 ? c->buf[scratch] : nullptr;
    if (!tmp) {
        const qlga_status st = ensure_scratch(c, bytes);
        if (st != QLGA_OK) return st;
        tmp = c->d_scratch;
    }
    cudaError_t e = launch_vorticity(L, storage_prec(c), c->buf[c->cur], tmp, c->nx, c->ny);
    if (e == cudaSuccess) e = cudaMemcpyAsync(omega, tmp, bytes, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_fail(c, "qlga_vorticity", e);
    return QLGA_OK;
}

// ---------------------------------------------------------------------------
// density, eq. (115), vortex detection
// ---------------------------------------------------------------------------
extern "C" qlga_status qlga_density(qlga_ctx* c, void* rho, int dst_on_device) {
    if (!c || !rho) return c ? fail(c, QLGA_EINVAL, "qlga_density: NULL") : QLGA_EINVAL;
    DeviceGuard guard(c);
    if (!c->have_state) return fail(c, QLGA_ESTATE, "qlga_density: no state set");
    Launch L{c->stream, &c->launches, c->device};
    const int64_t n = nsites(c);
    const size_t bytes = (size_t)n * real_size(c->prec);
    if (dst_on_device) {
        CU(c, launch_density(L, storage_prec(c), c->buf[c->cur], rho, n));
        return QLGA_OK;
    }
    const qlga_status st = ensure_scratch(c, bytes);
    if (st != QLGA_OK) return st;
    void* tmp = c->d_scratch;
    cudaError_t e = launch_density(L, storage_prec(c), c->buf[c->cur], tmp, n);
    if (e == cudaSuccess) e = cudaMemcpyAsync(rho, tmp, bytes, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_fail(c, "qlga_density", e);
    return QLGA_OK;
}

extern "C" qlga_status qlga_density_l2_error(qlga_ctx* c, const void* rho_ref, int src_on_device, double* host_eps) {
    if (!c || !rho_ref || !host_eps) return c ? fail(c, QLGA_EINVAL, "qlga_density_l2_error: NULL") : QLGA_EINVAL;
    DeviceGuard guard(c);
    if (!c->have_state) return fail(c, QLGA_ESTATE, "qlga_density_l2_error: no state set");
    Launch L{c->stream, &c->launches, c->device};
    const int64_t n = nsites(c);
    const size_t bytes = (size_t)n * real_size(c->prec);
    const void* ref = rho_ref;
    if (!src_on_device) {
        const qlga_status st = ensure_scratch(c, bytes);
        if (st != QLGA_OK) return st;
        cudaError_t e0 = cudaMemcpyAsync(c->d_scratch, rho_ref, bytes, cudaMemcpyHostToDevice, c->stream);
        if (e0 != cudaSuccess) return cuda_fail(c, "qlga_density_l2_error: H2D", e0);
        ref = c->d_scratch;
    }
    int blocks = c->obs_blocks;
    if ((int64_t)blocks * 256 > n) blocks = (int)((n + 255) / 256);
    double h = 0.0;
    cudaError_t e = launch_l2_error(L, storage_prec(c), c->buf[c->cur], ref, n, c->d_partials, blocks, c->d_sums);
    if (e == cudaSuccess) e = cudaMemcpyAsync(&h, c->d_sums, sizeof(double), cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_fail(c, "qlga_density_l2_error", e);
    *host_eps = h;
    return QLGA_OK;
}

extern "C" qlga_status qlga_vortices(qlga_ctx* c, int32_t* host_out, int64_t max_out, int64_t* host_count) {
    if (!c || !host_count || max_out < 0 || (max_out > 0 && !host_out))
        return c ? fail(c, QLGA_EINVAL, "qlga_vortices: bad arguments") : QLGA_EINVAL;
    DeviceGuard guard(c);
    if (c->ndim != 2) return fail(c, QLGA_EUNSUP, "qlga_vortices: 2D lattices only");
    if (!c->have_state) return fail(c, QLGA_ESTATE, "qlga_vortices: no state set");
    Launch L{c->stream, &c->launches, c->device};
    // scratch layout: [counter (16 bytes)][records]
    const size_t lbytes = (size_t)(max_out > 0 ? max_out : 1) * 4 * sizeof(int);
    const qlga_status sst = ensure_scratch(c, 16 + lbytes);
    if (sst != QLGA_OK) return sst;
    unsigned long long* counter = (unsigned long long*)c->d_scratch;
    int* list = (int*)((char*)c->d_scratch + 16);
    unsigned long long hc = 0;
    cudaError_t e = cudaMemsetAsync(counter, 0, sizeof(unsigned long long), c->stream);
    if (e == cudaSuccess) e = launch_vortices(L, storage_prec(c), c->buf[c->cur], c->nx, c->ny, list, (long long)max_out, counter);
    if (e == cudaSuccess) e = cudaMemcpyAsync(&hc, counter, sizeof(hc), cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e == cudaSuccess && max_out > 0) {
        const unsigned long long ncopy = hc < (unsigned long long)max_out ? hc : (unsigned long long)max_out;
        if (ncopy) e = cudaMemcpyAsync(host_out, list, (size_t)ncopy * 4 * sizeof(int), cudaMemcpyDeviceToHost, c->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    }
    if (e != cudaSuccess) return cuda_fail(c, "qlga_vortices", e);
    *host_count = (int64_t)hc;
    return QLGA_OK;
}

// ---------------------------------------------------------------------------
// Vortex tracking: association of two detections (qlga_track.cu)
// ---------------------------------------------------------------------------
extern "C" qlga_status qlga_vortex_match(qlga_ctx* c, const int32_t* host_prev, int64_t n_prev,
                                         const int32_t* host_cur, int64_t n_cur, int64_t max_dist2,
                                         int32_t* host_match_cur, int32_t* host_match_prev) {
    if (!c) return QLGA_EINVAL;
    if (n_prev < 0 || n_cur < 0 || n_prev > QLGA_MATCH_MAX || n_cur > QLGA_MATCH_MAX || max_dist2 < 0 ||
        (n_prev > 0 && (!host_prev || !host_match_prev)) || (n_cur > 0 && (!host_cur || !host_match_cur)))
        return fail(c, QLGA_EINVAL, "qlga_vortex_match: bad arguments (at most 65536 records per list)");
    DeviceGuard guard(c);
    if (c->ndim != 2) return fail(c, QLGA_EUNSUP, "qlga_vortex_match: 2D lattices only");
    if (c->nx > 2147483647LL || c->ny > 2147483647LL) return fail(c, QLGA_EUNSUP, "qlga_vortex_match: lattice too large");
    for (int64_t k = 0; k < n_prev + n_cur; ++k) {
        const int32_t* r = k < n_prev ? host_prev + 4 * k : host_cur + 4 * (k - n_prev);
        if (r[0] < 0 || r[0] > 4 || r[1] < 0 || r[1] >= c->nx || r[2] < 0 || r[2] >= c->ny)
            return fail(c, QLGA_EINVAL, "qlga_vortex_match: record outside the lattice");
    }
    if (n_prev + n_cur == 0) return QLGA_OK;
    // scratch: [prev records][cur records][nn_cur][nn_prev][match_cur][match_prev]
    const size_t rp = (size_t)n_prev * 16, rc = (size_t)n_cur * 16, ip = (size_t)n_prev * 4, ic = (size_t)n_cur * 4;
    const qlga_status st = ensure_scratch(c, rp + rc + 2 * (ip + ic) + 64);
    if (st != QLGA_OK) return st;
    char* base = (char*)c->d_scratch;
    int* d_prev = (int*)base; int* d_cur = (int*)(base + rp);
    int* nn_cur = (int*)(base + rp + rc); int* nn_prev = (int*)(base + rp + rc + ic);
    int* m_cur = (int*)(base + rp + rc + ic + ip); int* m_prev = (int*)(base + rp + rc + 2 * ic + ip);
    Launch L{c->stream, &c->launches, c->device};
    if (n_prev) CU(c, cudaMemcpyAsync(d_prev, host_prev, rp, cudaMemcpyHostToDevice, c->stream));
    if (n_cur) CU(c, cudaMemcpyAsync(d_cur, host_cur, rc, cudaMemcpyHostToDevice, c->stream));
    CU(c, launch_vortex_match(L, d_prev, (int)n_prev, d_cur, (int)n_cur, (int)c->nx, (int)c->ny, (long long)max_dist2,
                              nn_cur, nn_prev, m_cur, m_prev));
    if (n_cur) CU(c, cudaMemcpyAsync(host_match_cur, m_cur, ic, cudaMemcpyDeviceToHost, c->stream));
    if (n_prev) CU(c, cudaMemcpyAsync(host_match_prev, m_prev, ip, cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    return QLGA_OK;
}
