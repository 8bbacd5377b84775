// qlga_march.cu -- interaction-free strided pass by column marching (sm_100a).
//
// The four kinetic factors I'_{d,2} I'_{d,2} I'_{d,1} I'_{d,1} of a strided direction d (y, or z in 3D;
// eq. 107/108) act on every Zeeman level m separately and couple a site only to its two
// neighbours along d.  A pass that carries no interaction (the plain ordering's strided passes, eq. 108: U is
// applied once per step and rides on the x pass) is therefore a 1D radius-1 recurrence per (column, m): one
// thread takes one column of one level and marches along d, the four factors being the four stages of a
// register pipeline, each one row behind the one before it:
//
//     arrival of row r at a stage (a = the streamed component, b = the other one, messages as in qlga_math.cuh):
//         Fw = i a + b,  Bw = a + i b
//         emit row r-1:  a'(r-1) (kept from the last arrival),  b'(r-1) = Bw(r) - i Fw(r-1)
//         keep:          a'(r) = Fw(r-1) - i Bw(r),  Fw(r)
//
// No barrier, no exchange between threads; a warp reads 32 consecutive columns of one plane
// (512 contiguous bytes in fp64); per row a thread moves 2 x 16 bytes in and out and does 32 additions: the
// pass is bound by HBM.  A thread marches over a segment of the line plus 4 rows of run-in and run-out (the
// pipeline's depth), prefetching PF rows ahead with cp.async into a shared-memory ring that only it reads.  The arithmetic is the tile kernel's, operation for
// operation (same messages, same order, deferred halvings, one final scaling): the results are bit-identical.
#include "qlga_internal.h"

namespace qlga {

template <typename S>
struct MarchArgs {
    const typename vec2<S>::type* src;
    typename vec2<S>::type* dst;
    int64_t ncol;          // contiguous extent (x; x*y for the z pass)
    int64_t len;           // sites along the line
    int64_t stride;        // elements between consecutive sites of a line
    int64_t outer_stride;  // elements between consecutive outer indices (blockIdx.z)
    int64_t nsites;        // elements per plane of src
    int64_t dst_nsites;    // elements per plane of dst (= nsites unless dst is a band buffer)
    int64_t row0, row1;    // output rows [row0, row1) of the line (the whole line, or one band of it)
    int64_t dst_row_origin;// row r of the line is row r - dst_row_origin of dst
    int64_t seg;           // rows per segment
    int nseg;
    double out_scale;
#ifdef QLGA_TRACE
    unsigned long long* trace; int trace_id;
#endif
};
#ifdef QLGA_TRACE
__device__ __forceinline__ unsigned long long gtimer_m() { unsigned long long t; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t)); return t; }
#endif

template <typename T> struct MarchStage { cx<T> F, aP; };

// one factor of the pipeline: takes row r of its input, returns row r-1 of its output
template <typename T>
__device__ __forceinline__ void march_stage(MarchStage<T>& st, cx<T>& a, cx<T>& b) {
    const cx<T> Fw = add_i(b, a);              // i a + b  -> travels to r+e
    const cx<T> Bw = add_i(a, b);              // a + i b  -> travels to r-e
    const cx<T> a_out = st.aP;
    const cx<T> b_out = sub_i(Bw, st.F);       // b'(r-1) = Bw(r) - i Fw(r-1)
    st.aP = sub_i(st.F, Bw);                   // a'(r)   = Fw(r-1) - i Bw(r)
    st.F = Fw;
    a = a_out; b = b_out;
}

// one element of the state, global -> shared, asynchronously (16 bytes fp64 storage, 8 bytes fp32 storage)
__device__ __forceinline__ void cp_async_elem(double2* sm, const double2* g) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(sm)), "l"(g) : "memory");
}
__device__ __forceinline__ void cp_async_elem(float2* sm, const float2* g) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(sm)), "l"(g) : "memory");
}

#ifndef QLGA_MARCH_PF
#define QLGA_MARCH_PF 8
#endif
#ifndef QLGA_MARCH_MINB
#define QLGA_MARCH_MINB 1
#endif
template <typename T, typename S, int PF>
__global__ void __launch_bounds__(128, QLGA_MARCH_MINB) march_kernel(const __grid_constant__ MarchArgs<S> A) {
    using VS = typename vec2<S>::type;
#ifdef QLGA_TRACE
    if (A.trace && threadIdx.x == 0) atomicMin(&A.trace[2 * A.trace_id], gtimer_m());
#endif
    const int64_t x = (int64_t)blockIdx.x * 128 + threadIdx.x;
    if (x >= A.ncol) return;
    // level slowest: the CTAs resident at one time work on the same pair of planes (fewer concurrent DRAM streams:
    // measured 6.5-6.7 TB/s against 6.0-6.2 for a copy kernel of this access pattern)
    const int j = blockIdx.y / A.nseg;
    const int64_t sg = blockIdx.y % A.nseg;
    const int64_t s0 = A.row0 + sg * A.seg;
    const int64_t s1 = (s0 + A.seg < A.row1) ? s0 + A.seg : A.row1;   // output rows [s0, s1)
    const int64_t base = (int64_t)(2 * j) * A.nsites + (int64_t)blockIdx.z * A.outer_stride + x;
    const int64_t base_dst = (int64_t)(2 * j) * A.dst_nsites + (int64_t)blockIdx.z * A.outer_stride + x;
    const T scale = (T)A.out_scale;

    // input rows r0 .. r1-1 (periodic), r0 = s0 - 4, r1 = s1 + 4; the load pointer walks down the line and wraps.
    // Prefetch: every thread copies its own two elements of the next PF rows global -> shared with cp.async
    // (LDGSTS: no registers held by loads in flight, so 5-6 CTAs per SM keep ~200 KB in flight) and reads back
    // only what it copied itself -- no barrier.
    extern __shared__ __align__(16) unsigned char march_smem[];
    VS* ring = reinterpret_cast<VS*>(march_smem) + threadIdx.x;       // slot (u, component): ring[(2 u + component) * 128]
    const int64_t r0 = s0 - 4;
    const int nrows = (int)(s1 - s0) + 8;
    int64_t rl = r0 % A.len; if (rl < 0) rl += A.len;
    const VS* __restrict__ pl = A.src + base + rl * A.stride;          // component 1; component 2 is one plane further
    const VS* __restrict__ pl_wrap = A.src + base;
    int64_t to_wrap = A.len - rl;                                     // rows until the pointer wraps to row 0
    VS* __restrict__ ps = A.dst + base_dst + (s0 - A.dst_row_origin) * A.stride;                // store pointer (no wrap: s0 .. s1-1)
    int nload = nrows;
#pragma unroll
    for (int u = 0; u < PF; ++u) {
        if (nload > 0) {
            cp_async_elem(ring + (2 * u) * 128, pl);
            cp_async_elem(ring + (2 * u + 1) * 128, pl + A.nsites);
            pl += A.stride; --nload;
            if (--to_wrap == 0) { pl = pl_wrap; to_wrap = A.len; }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    }
    MarchStage<T> st[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) { st[k].F = mk<T>((T)0, (T)0); st[k].aP = mk<T>((T)0, (T)0); }

    int done = 0;                                                     // rows taken from the prefetch slots so far
    while (done < nrows) {
#pragma unroll
        for (int u = 0; u < PF; ++u) {
            if (done < nrows) {
                asm volatile("cp.async.wait_group %0;" ::"n"(PF - 1) : "memory");      // the oldest group has landed
                cx<T> c1 = ld_state<T, S>(ring + (2 * u) * 128);                       // spinor components 1, 2 of the row
                cx<T> c2 = ld_state<T, S>(ring + (2 * u + 1) * 128);
                if (nload > 0) {                               // refill the slot
                    cp_async_elem(ring + (2 * u) * 128, pl);
                    cp_async_elem(ring + (2 * u + 1) * 128, pl + A.nsites);
                    pl += A.stride; --nload;
                    if (--to_wrap == 0) { pl = pl_wrap; to_wrap = A.len; }
                }
                asm volatile("cp.async.commit_group;" ::: "memory");
                // factors in the order of eq. (108), rightmost first: component 2 streams twice, then component 1
                march_stage<T>(st[0], c2, c1);
                march_stage<T>(st[1], c2, c1);
                march_stage<T>(st[2], c1, c2);
                march_stage<T>(st[3], c1, c2);
                if (done >= 8) {                               // the row that leaves the pipeline: r - 4 >= s0
                    st_state<T, S>(ps, rmul(scale, c1));
                    st_state<T, S>(ps + A.dst_nsites, rmul(scale, c2));
                    ps += A.stride;
                }
                ++done;
            }
        }
    }
#ifdef QLGA_TRACE
    if (A.trace && threadIdx.x == 0) atomicMax(&A.trace[2 * A.trace_id + 1], gtimer_m());
#endif
}

template <typename T, typename S>
static cudaError_t run_march(const Launch& L, const PassParams& P, int dir) {
    MarchArgs<S> A;
    A.src = (const typename vec2<S>::type*)P.src;
    A.dst = (typename vec2<S>::type*)P.dst;
    A.nsites = P.src_plane ? P.src_plane : P.nx * P.ny * P.nz;
    A.dst_nsites = P.dst_plane ? P.dst_plane : P.nx * P.ny * P.nz;
    A.out_scale = P.out_scale;
#ifdef QLGA_TRACE
    A.trace = P.trace; A.trace_id = P.trace_id;
#endif
    int64_t n_outer;
    if (dir == 1) { A.ncol = P.nx; A.len = P.ny; A.stride = P.nx; n_outer = P.nz; A.outer_stride = P.nx * P.ny; }
    else          { A.ncol = P.nx * P.ny; A.len = P.nz; A.stride = P.nx * P.ny; n_outer = 1; A.outer_stride = 0; }
    // segments: about six waves of threads at full residency, at least 32 rows each (run-in and run-out cost 8)
    A.row0 = P.row_begin; A.row1 = P.row_end > P.row_begin ? P.row_end : A.len; A.dst_row_origin = P.dst_row_origin;
    const int64_t rows = A.row1 - A.row0;
    const int64_t per_seg = A.ncol * 5 * n_outer;
    int64_t nseg = (int64_t)(1400000 + per_seg - 1) / per_seg;
    if (nseg > rows / 32) nseg = rows / 32;
    if (nseg < 1) nseg = 1;
    A.seg = (rows + nseg - 1) / nseg;
    nseg = (rows + A.seg - 1) / A.seg;
    A.nseg = (int)nseg;
    const int64_t bx = (A.ncol + 127) / 128;
    if (bx > 2147483647LL || nseg * 5 > 65535 || n_outer > 65535) return cudaErrorInvalidValue;
    dim3 grid((unsigned)bx, (unsigned)(5 * nseg), (unsigned)n_outer);
    constexpr size_t smem = (size_t)QLGA_MARCH_PF * 2 * 128 * sizeof(typename vec2<S>::type);
    static_assert(smem <= 48 * 1024, "prefetch ring beyond the default dynamic shared memory");
    march_kernel<T, S, QLGA_MARCH_PF><<<grid, 128, smem, L.stream>>>(A);
    ++*L.counter;
    return cudaGetLastError();
}

bool march_supported(int dir, const PassParams& P) {
    if (dir != 1 && dir != 2) return false;
    if (P.umode != 0 || P.utail != 0 || P.ksteps != 1) return false;
    const int64_t n_outer = (dir == 1) ? P.nz : 1;
    const int64_t len = (dir == 1) ? P.ny : P.nz;
    return n_outer <= 65535 && len >= 1;
}

cudaError_t launch_march(const Launch& L, qlga_prec prec, int dir, const PassParams& P) {
    switch (prec) {
        case QLGA_F64: return run_march<double, double>(L, P, dir);
        case QLGA_F32: return run_march<float, float>(L, P, dir);
        case QLGA_F32X: return run_march<double, float>(L, P, dir);
    }
    return cudaErrorInvalidValue;
}

}  // namespace qlga
