// qlga_step.cu -- fp64 instantiation of the fused pass kernels (qlga_pass.cuh), the precision
// dispatch of the pass launcher and the per-operator cross-check kernels.
#include "qlga_pass.cuh"

namespace qlga {

int max_ksteps(int threads) { return (threads - 8) / 8; }

// the (direction, CTA size, columns) combinations launch_pass_t has an instantiation for (0 = default)
bool pass_tile_supported(int dir, int threads, int cx) {
    if (dir == 0) return threads == 0 || threads == 64 || threads == 96 || threads == 128 || threads == 192 || threads == 256;
    if (cx == 0 && threads == 0) return true;
    if (cx == 0) return threads == 128 || threads == 192;           // fp64 default 1 column, fp32 2: both have 128 and 192
    if (threads == 0) return cx == 1 || cx == 2 || cx == 4 || cx == 8;
    switch (cx * 1000 + threads) {
        case 1064: case 1096: case 1128: case 1192: case 2128: case 2192: case 2256: case 4256: case 8256: return true;
        default: return false;
    }
}

cudaError_t launch_pass_f64(const Launch& L, int dir, const PassParams& P, int threads, int cxw) {
    return launch_pass_t<double, double>(L, dir, P, threads, cxw);
}

cudaError_t launch_pass(const Launch& L, qlga_prec prec, int dir, const PassParams& P,
                        int threads, int cxw) {
    switch (prec) {
        case QLGA_F64: return launch_pass_f64(L, dir, P, threads, cxw);
        case QLGA_F32: return launch_pass_f32(L, dir, P, threads, cxw);
        case QLGA_F32X: return launch_pass_mixed(L, dir, P, threads, cxw);
    }
    return cudaErrorInvalidValue;
}

// ---------------------------------------------------------------------------
// One kernel per operator: U in place, I'_{d,sigma} out of place straight from
// global memory.  Slow (one HBM round trip per operator); kept as the GPU-side
// cross-check of the fused passes and selectable with QLGA_OPT_PATH = 1.
// ---------------------------------------------------------------------------
template <typename T, typename S>
__global__ void __launch_bounds__(128) interaction_kernel(typename vec2<S>::type* q, int64_t n,
                                                          UConst<T> uc, const __grid_constant__ ExpTable tab, int* flag) {
    // every thread of the CTA takes part (the order selection is a warp reduction);
    // threads past the end work on a copy of the last site and do not store
    int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool ok = r < n;
    if (!ok) r = n - 1;
    Site<T> s;
#pragma unroll
    for (int j = 0; j < 5; ++j)
#pragma unroll
        for (int sg = 0; sg < 2; ++sg) s.q[j][sg] = ld_state<T, S>(q + (int64_t)(2 * j + sg) * n + r);
    interaction<T>(s, uc, tab, flag);
    if (ok) {
#pragma unroll
        for (int j = 0; j < 5; ++j)
#pragma unroll
            for (int sg = 0; sg < 2; ++sg) st_state<T, S>(q + (int64_t)(2 * j + sg) * n + r, s.q[j][sg]);
    }
}

template <typename T, typename S>
__global__ void __launch_bounds__(128) kinetic_kernel(const typename vec2<S>::type* src,
                                                      typename vec2<S>::type* dst,
                                                      int64_t nx, int64_t ny, int64_t nz, int dir, int sigma) {
    using V = typename vec2<T>::type;
    using VS = typename vec2<S>::type;
    const int64_t n = nx * ny * nz;
    const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n) return;
    const int64_t x = r % nx, y = (r / nx) % ny, z = r / (nx * ny);
    int64_t rm, rp;
    if (dir == 0) {
        rm = r - x + (x == 0 ? nx - 1 : x - 1);
        rp = r - x + (x == nx - 1 ? 0 : x + 1);
    } else if (dir == 1) {
        rm = r + ((y == 0 ? ny - 1 : y - 1) - y) * nx;
        rp = r + ((y == ny - 1 ? 0 : y + 1) - y) * nx;
    } else {
        rm = r + ((z == 0 ? nz - 1 : z - 1) - z) * nx * ny;
        rp = r + ((z == nz - 1 ? 0 : z + 1) - z) * nx * ny;
    }
    const T half = (T)0.5;
    for (int j = 0; j < 5; ++j) {
        const VS* pa = src + (int64_t)(2 * j + sigma) * n;
        const VS* pb = src + (int64_t)(2 * j + 1 - sigma) * n;
        const cx<T> a = ld_state<T, S>(pa + r), b = ld_state<T, S>(pb + r), am = ld_state<T, S>(pa + rm),
                    bm = ld_state<T, S>(pb + rm), ap = ld_state<T, S>(pa + rp), bp = ld_state<T, S>(pb + rp);
        // a'(r) = (1/2)[-i a + b + i a(r-e) + b(r-e)],  b'(r) = (1/2)[a(r+e) + i b(r+e) + a - i b]
        cx<T> za, zb;
        za.re = half * ((a.im + b.re) + (bm.re - am.im));
        za.im = half * ((b.im - a.re) + (am.re + bm.im));
        zb.re = half * ((ap.re - bp.im) + (a.re + b.im));
        zb.im = half * ((ap.im + bp.re) + (a.im - b.re));
        st_state<T, S>(dst + (int64_t)(2 * j + sigma) * n + r, za);
        st_state<T, S>(dst + (int64_t)(2 * j + 1 - sigma) * n + r, zb);
    }
}

cudaError_t launch_interaction(const Launch& L, qlga_prec prec, void* q, int64_t n,
                               const double g[3], double smu, const ExpTable& tab, int* flag) {
    const unsigned blocks = (unsigned)((n + 127) / 128);
    if (prec == QLGA_F32) {
        UConst<float> uc = make_uconst<float>(g[0], g[1], g[2], smu);
        interaction_kernel<float, float><<<blocks, 128, 0, L.stream>>>((float2*)q, n, uc, tab, flag);
    } else {
        UConst<double> uc = make_uconst<double>(g[0], g[1], g[2], smu);
        if (prec == QLGA_F64) interaction_kernel<double, double><<<blocks, 128, 0, L.stream>>>((double2*)q, n, uc, tab, flag);
        else interaction_kernel<double, float><<<blocks, 128, 0, L.stream>>>((float2*)q, n, uc, tab, flag);
    }
    ++*L.counter;
    return cudaGetLastError();
}

cudaError_t launch_kinetic(const Launch& L, qlga_prec prec, const void* src, void* dst,
                           int64_t nx, int64_t ny, int64_t nz, int dir, int sigma) {
    const int64_t n = nx * ny * nz;
    const unsigned blocks = (unsigned)((n + 127) / 128);
    if (prec == QLGA_F64)
        kinetic_kernel<double, double><<<blocks, 128, 0, L.stream>>>((const double2*)src, (double2*)dst, nx, ny, nz, dir, sigma);
    else if (prec == QLGA_F32)
        kinetic_kernel<float, float><<<blocks, 128, 0, L.stream>>>((const float2*)src, (float2*)dst, nx, ny, nz, dir, sigma);
    else
        kinetic_kernel<double, float><<<blocks, 128, 0, L.stream>>>((const float2*)src, (float2*)dst, nx, ny, nz, dir, sigma);
    ++*L.counter;
    return cudaGetLastError();
}

}  // namespace qlga
