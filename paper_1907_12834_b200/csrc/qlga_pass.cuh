// qlga_pass.cuh -- the fused directional pass kernel of the QLGA time step (sm_100a), as a
// template over the arithmetic type T and the storage type S.  Instantiated in
//   qlga_step.cu       T = S = double          (QLGA_F64)
//   qlga_step_f32.cu   T = S = float           (QLGA_F32)
//   qlga_step_mixed.cu T = double, S = float   (QLGA_F32X: fp32 storage, fp64 arithmetic in registers)
// so that the three sets compile in parallel.
//
// One pass = the four kinetic factors of one lattice direction,
//     I'_{d,1} I'_{d,1} I'_{d,2} I'_{d,2}          (eq. 108 / 112)
// with the interaction U interleaved before every factor (eq. 112), before the
// first factor only (eq. 108: U is the rightmost operator of the step), after the last
// factor (plain ordering: the next step's U), or not at all.  A 1D step is one x pass; a
// 2D step is a y pass followed by an x pass (R7); 3D: z, y, x.
//
// Design: one lattice site per thread, the 10 complex
// amplitudes live in registers for the whole pass.  A CTA owns a line of TS sites
// along the pass direction (x pass) or CX adjacent such lines (strided passes: CX columns,
// so a warp reads CX*16 B contiguous segments).  The only neighbour traffic of a
// kinetic factor is one 5-vector to the site at r+e and one to r-e; it moves through
// shared memory (128-bit, conflict free, double buffered: one barrier per factor).
// Lines overlap by a halo of 4 sites per fused time step on each side and the halo
// threads recompute ((TS-8)/TS efficiency); nothing but the final state goes back to
// HBM: 320 B per site per pass in fp64.
#pragma once
#include <atomic>
#include "qlga_internal.h"

namespace qlga {

template <typename T, typename S>
struct PassArgs {
    const typename vec2<S>::type* src;
    typename vec2<S>::type* dst;
    // geometry of the pass: sites along a line are `stride` elements apart and `len` many;
    // `nx` columns (x, unit stride) and `n_outer` outer indices (`outer_stride` apart) give
    // the lines.  x pass: len = nx, the lines are the ny*nz rows (outer_stride = nx).
    // y pass: stride = nx, len = ny, outer = z.   z pass: stride = nx*ny, len = nz, outer = y.
    int64_t nx, len, stride, n_outer, outer_stride, nsites;
    int64_t nsites_dst;         // plane stride of dst (= nsites unless dst is another view of the lattice: band mode)
    int ksteps, umode, utail;
    UConst<T> uc[4];
    UConst<T> uct;              // trailing U of the plain ordering (see pass_kernel)
    T out_scale;
    int* flag;                  // device error word (qlga_internal.h, FLAG_*)
    ExpTable tab;
#ifdef QLGA_TRACE
    unsigned long long* trace; int trace_id;
#endif
};

#ifdef QLGA_TRACE
__device__ __forceinline__ unsigned long long gtimer() { unsigned long long t; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t)); return t; }
#endif

__device__ __forceinline__ int64_t pmod(int64_t a, int64_t n) {
    int64_t r = a % n;
    return r < 0 ? r + n : r;
}

__device__ __forceinline__ void st_shared(double2* p, cx<double> z) { *reinterpret_cast<cx<double>*>(p) = z; }
__device__ __forceinline__ void st_shared(float2* p, cx<float> z) {
    asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"((unsigned)__cvta_generic_to_shared(p)), "f"(z.re), "f"(z.im) : "memory");
}

// One kinetic factor I'_{d,SIGMA} of the pass, preceded by the interaction if the
// ordering asks for it.  SIGMA (compile time) = the spinor component that streams.
// The two message 5-vectors of a site go to its neighbours along the line through
// shared memory, one 16-byte (8-byte in fp32) element per thread and plane
// ([j][thread]: conflict free), double buffered so that one barrier per factor
// suffices.  (A warp-shuffle exchange was measured first: SHFL.32 issues at 6 cycles
// per warp on sm_100a and a factor needs 40 of them.)
template <typename T, typename S, int CX, int NT, int SIGMA, bool HASU>
__device__ __forceinline__ void factor(Site<T>& s, const PassArgs<T, S>& P, int f, int t, int& pb,
                                       typename vec2<T>::type (*sF)[5][NT], typename vec2<T>::type (*sB)[5][NT]) {
    using V = typename vec2<T>::type;
    if constexpr (HASU) {
        if (P.umode == 2 || (P.umode == 1 && f == 0)) interaction<T>(s, P.uc[f], P.tab, P.flag);
    }

    cx<T> Fw[5], Bw[5], Fp[5], Bn[5];
    kin_messages<T>(s, SIGMA, Fw, Bw);
#pragma unroll
    for (int j = 0; j < 5; ++j) {
        st_shared(&sF[pb][j][t], Fw[j]);
        st_shared(&sB[pb][j][t], Bw[j]);
    }
    __syncthreads();
    // the first / last CX threads of the CTA have no neighbour in the tile: they are halo
    // threads whose values are never stored; they read their own slot
    const int tm = (t >= CX) ? t - CX : t;
    const int tp = (t + CX < NT) ? t + CX : t;
#pragma unroll
    for (int j = 0; j < 5; ++j) {
        Fp[j] = *reinterpret_cast<const cx<T>*>(&sF[pb][j][tm]);
        Bn[j] = *reinterpret_cast<const cx<T>*>(&sB[pb][j][tp]);
    }
    pb ^= 1;
    kin_update<T>(s, SIGMA, Fw, Bw, Fp, Bn);
}

// experiment knobs (compile time)
#ifndef QLGA_MINB128
#define QLGA_MINB128 3
#endif
// fp32 is latency bound at 4 CTAs per SM (ncu: FMA pipe 62 %, issue 67 % busy): a few spilled
// words buy 5 CTAs per SM (96 registers): 8192^2 interleaved 3.90 -> 4.3 GSUP/s.  (6 CTAs, 80
// registers, was faster for the x pass while it spilled 24 bytes and slower once it spilled 172.)
#ifndef QLGA_MINB128_F32
#define QLGA_MINB128_F32 5
#endif
#ifndef QLGA_MINB256_NOU
#define QLGA_MINB256_NOU 2
#endif
#ifndef QLGA_MINB_NOU
#define QLGA_MINB_NOU 4
#endif
#ifndef QLGA_MINB128_F32X
#define QLGA_MINB128_F32X 5
#endif

// HASU = false: a pass without any interaction (the plain ordering's later passes): the same
// kernel minus the interaction code, a third of the registers, so more CTAs per SM keep the
// HBM pipe full (this pass is memory-bound).
template <typename T, typename S, int DIR, int CX, int NT, bool HASU>
__global__ void __launch_bounds__(NT, (HASU ? (NT >= 192 ? 2 : (NT >= 128 ? (sizeof(T) == 8 ? QLGA_MINB128 : (DIR == 0 ? QLGA_MINB128_F32X : QLGA_MINB128_F32))
                                                                         : (NT >= 96 ? 4 : 6)))
                                            : (NT >= 256 ? QLGA_MINB256_NOU : (NT >= 192 ? 2 : QLGA_MINB_NOU))))
pass_kernel(const __grid_constant__ PassArgs<T, S> P) {
    using V = typename vec2<T>::type;
    constexpr int TS = NT / CX;              // sites per line handled by the CTA
    static_assert(NT % 32 == 0 && 32 % CX == 0 && CX < 32, "bad tile");
    static_assert(DIR == 1 || CX == 1, "x pass uses one line per CTA");

    extern __shared__ __align__(16) unsigned char smem_raw[];
    V (*sF)[5][NT] = reinterpret_cast<V (*)[5][NT]>(smem_raw);
    V (*sB)[5][NT] = sF + 2;

    const int t = threadIdx.x;
#ifdef QLGA_TRACE
    if (P.trace && t == 0) atomicMin(&P.trace[2 * P.trace_id], gtimer());
#endif
    const int c = t % CX, i = t / CX;
    const int H = 4 * P.ksteps;
    const int wout = TS - 2 * H;
    const int64_t n = P.nsites;

    int64_t spos, idx;
    const int64_t extent = P.len;
    bool col_ok = true;
    if (DIR == 0) {
        const int64_t tiles = (P.len + wout - 1) / wout;
        const int64_t tile = blockIdx.x % tiles;
        const int64_t row = blockIdx.x / tiles;
        spos = tile * wout - H + i;
        idx = row * P.outer_stride + pmod(spos, P.len);
    } else {
        const int64_t tiles_c = (P.nx + CX - 1) / CX;
        const int64_t tiles_s = (P.len + wout - 1) / wout;
        const int64_t tc = blockIdx.x % tiles_c;
        const int64_t rest = blockIdx.x / tiles_c;
        const int64_t ts = rest % tiles_s;
        const int64_t outer = rest / tiles_s;
        int64_t x = tc * CX + c;
        col_ok = x < P.nx;
        if (!col_ok) x = P.nx - 1;
        spos = ts * wout - H + i;
        idx = outer * P.outer_stride + pmod(spos, P.len) * P.stride + x;
    }

    // s.q[j][sigma]: sigma = 0,1 <-> spinor component 1,2 (the planes' own order)
    Site<T> s;
#pragma unroll
    for (int j = 0; j < 5; ++j) {
        s.q[j][0] = ld_state<T, S>(P.src + (int64_t)(2 * j + 0) * n + idx);
        s.q[j][1] = ld_state<T, S>(P.src + (int64_t)(2 * j + 1) * n + idx);
    }

    int pb = 0;
#pragma unroll 1
    for (int st = 0; st < P.ksteps; ++st) {
        // factors I'_{d,2} I'_{d,2} then I'_{d,1} I'_{d,1} (rightmost first): two code instances,
        // one per streamed component, so that no register ever changes role
#pragma unroll 1
        for (int f = 0; f < 2; ++f)
            factor<T, S, CX, NT, 1, HASU>(s, P, f, t, pb, sF, sB);
#pragma unroll 1
        for (int f = 2; f < 4; ++f)
            factor<T, S, CX, NT, 0, HASU>(s, P, f, t, pb, sF, sB);
        // undo the four deferred halvings (exact)
#pragma unroll
        for (int j = 0; j < 5; ++j) {
            s.q[j][0] = rmul(P.out_scale, s.q[j][0]);
            s.q[j][1] = rmul(P.out_scale, s.q[j][1]);
        }
    }
    // Plain ordering, several steps per call: the next step's U (the rightmost operator of eq. 108) is
    // applied here, at the end of the last pass of this step, where the state is final and in registers
    // and the pass is otherwise memory-bound -- instead of at the start of the next step's first pass,
    // where the halo threads would recompute it.  Site-local, so the product of operators is the same.
    if constexpr (HASU) {
        if (P.utail) interaction<T>(s, P.uct, P.tab, P.flag);
    }

    if (i >= H && i < TS - H && spos < extent && col_ok) {
#pragma unroll
        for (int j = 0; j < 5; ++j) {
            st_state<T, S>(P.dst + (int64_t)(2 * j + 0) * P.nsites_dst + idx, s.q[j][0]);
            st_state<T, S>(P.dst + (int64_t)(2 * j + 1) * P.nsites_dst + idx, s.q[j][1]);
        }
    }
#ifdef QLGA_TRACE
    if (P.trace && t == 0) atomicMax(&P.trace[2 * P.trace_id + 1], gtimer());
#endif
}

template <typename T, typename S>
static PassArgs<T, S> make_args(const PassParams& P, int dir) {
    PassArgs<T, S> A;
    A.src = (const typename vec2<S>::type*)P.src;
    A.dst = (typename vec2<S>::type*)P.dst;
    A.flag = P.flag;
    A.nx = P.nx; A.nsites = P.src_plane ? P.src_plane : P.nx * P.ny * P.nz;
    A.nsites_dst = P.dst_plane ? P.dst_plane : P.nx * P.ny * P.nz; A.ksteps = P.ksteps; A.umode = P.umode; A.utail = P.utail;
    A.uct = make_uconst<T>(P.gt[0], P.gt[1], P.gt[2], P.smu);
    for (int f = 0; f < 4; ++f) A.uc[f] = make_uconst<T>(P.g[f][0], P.g[f][1], P.g[f][2], P.smu);
    A.out_scale = (T)P.out_scale;
    A.tab = P.tab;
#ifdef QLGA_TRACE
    A.trace = P.trace; A.trace_id = P.trace_id;
#endif
    if (dir == 0)      { A.len = P.nx; A.stride = 1;           A.n_outer = P.ny * P.nz; A.outer_stride = P.nx; }
    else if (dir == 1) { A.len = P.ny; A.stride = P.nx;        A.n_outer = P.nz;        A.outer_stride = P.nx * P.ny; }
    else               { A.len = P.nz; A.stride = P.nx * P.ny; A.n_outer = P.ny;        A.outer_stride = P.nx; }
    return A;
}

template <typename T, typename S, int DIR, int CX, int NT>
static cudaError_t run_pass(const Launch& L, const PassParams& P, int dir) {
    constexpr int TS = NT / CX;
    const int wout = TS - 8 * P.ksteps;
    if (wout <= 0) return cudaErrorInvalidValue;
    PassArgs<T, S> A = make_args<T, S>(P, dir);
    int64_t blocks;
    if (DIR == 0) blocks = ((A.len + wout - 1) / wout) * A.n_outer;
    else blocks = ((A.nx + CX - 1) / CX) * ((A.len + wout - 1) / wout) * A.n_outer;
    if (blocks <= 0 || blocks > 2147483647LL) return cudaErrorInvalidValue;
    constexpr size_t smem = (size_t)4 * 5 * NT * sizeof(typename vec2<T>::type);   // sF[2], sB[2]
    // more than 48 KB of dynamic shared memory needs an opt-in, which is a per-device attribute of the
    // function: one bit per device and instantiation (set once; a race only repeats the idempotent call)
    static std::atomic<uint64_t> configured{0};
    const uint64_t bit = 1ull << (L.device & 63);
    if (!(configured.load(std::memory_order_acquire) & bit)) {
        cudaError_t e = cudaFuncSetAttribute(pass_kernel<T, S, DIR, CX, NT, true>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(pass_kernel<T, S, DIR, CX, NT, false>,
                                     cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        if (L.device < 64) configured.fetch_or(bit, std::memory_order_release);
    }
    if (P.umode != 0 || P.utail) pass_kernel<T, S, DIR, CX, NT, true><<<(unsigned)blocks, NT, smem, L.stream>>>(A);
    else pass_kernel<T, S, DIR, CX, NT, false><<<(unsigned)blocks, NT, smem, L.stream>>>(A);
    ++*L.counter;
    return cudaGetLastError();
}

template <typename T, typename S>
static cudaError_t launch_pass_t(const Launch& L, int dir, const PassParams& P, int threads, int cxw) {
    if (dir == 0) {
        if (threads == 0) threads = 128;
        switch (threads) {
            case 64: return run_pass<T, S, 0, 1, 64>(L, P, dir);
            case 96: return run_pass<T, S, 0, 1, 96>(L, P, dir);
            case 128: return run_pass<T, S, 0, 1, 128>(L, P, dir);
            case 192: return run_pass<T, S, 0, 1, 192>(L, P, dir);
            case 256: return run_pass<T, S, 0, 1, 256>(L, P, dir);
            default: return cudaErrorInvalidValue;
        }
    }
    // defaults: fp64 is register-heavy and FP64-pipe bound: 128-thread CTAs (three per SM without
    // spills), one column x 128 rows (least halo recompute; the half-used 32-byte sectors are
    // completed by the neighbouring column's CTA out of L2); fp32 takes two columns x 64 rows
    // (measured at 8192^2: 8.65 ms against 8.80 for 4 x 64 and 10.3 for 1 x 128)
    if (cxw == 0) cxw = (sizeof(T) == 8) ? 1 : 2;
    if (threads == 0) threads = (cxw <= 2) ? 128 : 256;
    switch (cxw * 1000 + threads) {
        case 1064: return run_pass<T, S, 1, 1, 64>(L, P, dir);
        case 1096: return run_pass<T, S, 1, 1, 96>(L, P, dir);
        case 1128: return run_pass<T, S, 1, 1, 128>(L, P, dir);
        case 1192: return run_pass<T, S, 1, 1, 192>(L, P, dir);
        case 2128: return run_pass<T, S, 1, 2, 128>(L, P, dir);
        case 2192: return run_pass<T, S, 1, 2, 192>(L, P, dir);
        case 2256: return run_pass<T, S, 1, 2, 256>(L, P, dir);
        case 4256: return run_pass<T, S, 1, 4, 256>(L, P, dir);
        case 8256: return run_pass<T, S, 1, 8, 256>(L, P, dir);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace qlga
