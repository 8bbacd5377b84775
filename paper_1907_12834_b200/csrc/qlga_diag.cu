// qlga_diag.cu -- lattice reductions (observables), lattice vorticity and the
// psi <-> q conversions of the QLGA library (sm_100a).
//
// Observables: column-marching work units (see observables_kernel), 19 fp64 accumulators per
// thread (fp64 even for an fp32 state), warp-shuffle tree, one shared-memory tree per block,
// per-block partials to global memory and a second single-block pass -- deterministic, no
// atomics.  Definitions: include/qlga.h (eq. 3-5, 59-60, 85, 32 of PAPER.md).
#include "qlga_internal.h"

namespace qlga {

// accumulator slots
enum { A_N0 = 0, A_NQ = 5, A_FX = 6, A_FY = 7, A_FZ = 8, A_A00R = 9, A_A00I = 10, A_A2 = 11,
       A_EKIN = 12, A_RHO2 = 13, A_F2 = 14, A_OVR = 15, A_OVI = 16, A_SPARE0 = 17, A_SPARE1 = 18 };

template <typename T>
__device__ __forceinline__ void load_psi(const typename vec2<T>::type* q, int64_t n, int64_t r,
                                         double pr[5], double pi[5], double* normq) {
    double nq = 0.0;
#pragma unroll
    for (int j = 0; j < 5; ++j) {
        const typename vec2<T>::type a = q[(int64_t)(2 * j) * n + r], b = q[(int64_t)(2 * j + 1) * n + r];
        const double ar = a.x, ai = a.y, br = b.x, bi = b.y;
        pr[j] = ar + br; pi[j] = ai + bi;
        nq += ar * ar + ai * ai + br * br + bi * bi;
    }
    if (normq) *normq = nq;
}

// The sums of one site: psi = (pr, pi), |q|^2 = nq, the +x / +y / +z neighbours' psi, the previous state's psi.
__device__ __forceinline__ void obs_site(double acc[OBS_NACC], int ndim, bool has_prev, double nq,
                                         const double pr[5], const double pi[5], const double xr[5], const double xi[5],
                                         const double yr[5], const double yi[5], const double zr[5], const double zi[5],
                                         const double or_[5], const double oi[5]) {
    const double rt6 = 2.4494897427831780981972840747059;
    const double irt5 = 0.44721359549995793928183473374626;
    acc[A_NQ] += nq;
    double nm[5];
#pragma unroll
    for (int j = 0; j < 5; ++j) { nm[j] = pr[j] * pr[j] + pi[j] * pi[j]; acc[A_N0 + j] += nm[j]; }
    const double rho = nm[0] + nm[1] + nm[2] + nm[3] + nm[4];
    const double Fz = 2.0 * (nm[0] - nm[4]) + (nm[1] - nm[3]);
    // F_+ = 2(conj(psi_2) psi_1 + conj(psi_-1) psi_-2) + sqrt6 (conj(psi_1) psi_0 + conj(psi_0) psi_-1)
    const double far_ = pr[0] * pr[1] + pi[0] * pi[1] + pr[3] * pr[4] + pi[3] * pi[4];
    const double fai = pr[0] * pi[1] - pi[0] * pr[1] + pr[3] * pi[4] - pi[3] * pr[4];
    const double fbr = pr[1] * pr[2] + pi[1] * pi[2] + pr[2] * pr[3] + pi[2] * pi[3];
    const double fbi = pr[1] * pi[2] - pi[1] * pr[2] + pr[2] * pi[3] - pi[2] * pr[3];
    const double Fx = 2.0 * far_ + rt6 * fbr, Fy = 2.0 * fai + rt6 * fbi;
    acc[A_FX] += Fx; acc[A_FY] += Fy; acc[A_FZ] += Fz;
    // A00 = (2 psi_2 psi_-2 - 2 psi_1 psi_-1 + psi_0^2)/sqrt5
    const double tr = 2.0 * (pr[0] * pr[4] - pi[0] * pi[4]) - 2.0 * (pr[1] * pr[3] - pi[1] * pi[3])
            + (pr[2] * pr[2] - pi[2] * pi[2]);
    const double ti = 2.0 * (pr[0] * pi[4] + pi[0] * pr[4]) - 2.0 * (pr[1] * pi[3] + pi[1] * pr[3])
            + 2.0 * pr[2] * pi[2];
    const double ar = tr * irt5, ai = ti * irt5;
    acc[A_A00R] += ar; acc[A_A00I] += ai; acc[A_A2] += ar * ar + ai * ai;
    acc[A_RHO2] += rho * rho;
    acc[A_F2] += Fx * Fx + Fy * Fy + Fz * Fz;
    // kinetic: forward differences along x (and y, z)
#pragma unroll
    for (int j = 0; j < 5; ++j) {
        const double dr = xr[j] - pr[j], di = xi[j] - pi[j];
        acc[A_EKIN] += dr * dr + di * di;
    }
    if (ndim >= 2) {
#pragma unroll
        for (int j = 0; j < 5; ++j) {
            const double dr = yr[j] - pr[j], di = yi[j] - pi[j];
            acc[A_EKIN] += dr * dr + di * di;
        }
    }
    if (ndim == 3) {
#pragma unroll
        for (int j = 0; j < 5; ++j) {
            const double dr = zr[j] - pr[j], di = zi[j] - pi[j];
            acc[A_EKIN] += dr * dr + di * di;
        }
    }
    if (has_prev) {       // <psi(t)|psi(t - tau)>
#pragma unroll
        for (int j = 0; j < 5; ++j) {
            acc[A_OVR] += pr[j] * or_[j] + pi[j] * oi[j];
            acc[A_OVI] += pr[j] * oi[j] - pi[j] * or_[j];
        }
    }
}

// Work unit = 128 columns (x) x a segment of rows (y) of one z layer.  A thread owns one column of the unit and
// marches down its rows: every site's ten amplitudes are loaded once (the row below is kept in registers for the
// y difference of the kinetic energy; the +x neighbour is a load that hits the line its neighbour thread just
// fetched; the +z neighbour and the previous state are plain loads).  The first version re-read the +y neighbour
// through L2 for every site: 4.1 ms at 8192^2 (40 % of the copy bandwidth).
struct ObsGeom {
    int64_t nx, ny, nz;
    int ndim;
    int64_t x0, x1, y0, y1, z0, z1;       // the sites summed: [x0,x1) x [y0,y1) x [z0,z1)
    int64_t seg;                          // rows per unit
    int64_t ncb, nsg;                     // column blocks, segments; units = ncb * nsg * (z1 - z0)
};

template <typename T>
__global__ void __launch_bounds__(128, sizeof(T) == 8 ? 2 : 4) observables_kernel(const typename vec2<T>::type* __restrict__ q,
                                                          const typename vec2<T>::type* __restrict__ qprev,
                                                          const __grid_constant__ ObsGeom G, double* partials) {
    const int64_t n = G.nx * G.ny * G.nz;
    double acc[OBS_NACC];
#pragma unroll
    for (int k = 0; k < OBS_NACC; ++k) acc[k] = 0.0;
    const double rt6 = 2.4494897427831780981972840747059;
    const double irt5 = 0.44721359549995793928183473374626;

    const int64_t units = G.ncb * G.nsg * (G.z1 - G.z0);
    for (int64_t u = blockIdx.x; u < units; u += gridDim.x) {
        const int64_t cb = u % G.ncb, sg = (u / G.ncb) % G.nsg, z = G.z0 + u / (G.ncb * G.nsg);
        const int64_t x = G.x0 + cb * 128 + threadIdx.x;
        if (x >= G.x1) continue;
        const int64_t ys = G.y0 + sg * G.seg;
        const int64_t ye = (ys + G.seg < G.y1) ? ys + G.seg : G.y1;
        const int64_t xn = (x == G.nx - 1) ? 0 : x + 1;
        const int64_t zn = (z == G.nz - 1) ? 0 : z + 1;
        double pr[5], pi[5], nq;
        load_psi<T>(q, n, (z * G.ny + ys) * G.nx + x, pr, pi, &nq);
        for (int64_t y = ys; y < ye; ++y) {
            const int64_t row = (z * G.ny + y) * G.nx;
            // the loads of this row first: the row below, the +x (and +z) neighbour, the previous state
            double yr[5], yi[5], ynq = 0.0, xr[5], xi[5], zr[5], zi[5], or_[5], oi[5];
            const int64_t yn = (y == G.ny - 1) ? 0 : y + 1;
            if (G.ndim >= 2) load_psi<T>(q, n, (z * G.ny + yn) * G.nx + x, yr, yi, &ynq);
            load_psi<T>(q, n, row + xn, xr, xi, nullptr);
            if (G.ndim == 3) load_psi<T>(q, n, (zn * G.ny + y) * G.nx + x, zr, zi, nullptr);
            if (qprev) load_psi<T>(qprev, n, row + x, or_, oi, nullptr);

            obs_site(acc, G.ndim, qprev != nullptr, nq, pr, pi, xr, xi, yr, yi, zr, zi, or_, oi);
            // the row below becomes the current row
#pragma unroll
            for (int j = 0; j < 5; ++j) { pr[j] = yr[j]; pi[j] = yi[j]; }
            nq = ynq;
        }
    }

    __shared__ double sm[4][OBS_NACC];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < OBS_NACC; ++k) {
        double v = acc[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) sm[warp][k] = v;
    }
    __syncthreads();
    if (threadIdx.x < OBS_NACC) {
        double v = 0.0;
        for (int w = 0; w < 4; ++w) v += sm[w][threadIdx.x];
        partials[(int64_t)blockIdx.x * OBS_NACC + threadIdx.x] = v;
    }
}

// 2D lattices: the same work units with the loads staged through shared memory (round 2).  Every thread copies the ten
// amplitudes of its column, one row per cp.async group, R - 2 rows ahead of the row it sums (no registers held by loads
// in flight: 40 KB per CTA, 80 KB per SM in flight, against ~40 KB of the register version, which reached 58 % of the
// copy bandwidth at 250 registers); psi of the row below is formed once per site from the ring and handed to the left
// neighbour through a small double-buffered array (the +x difference of the next row), so a site costs 20 + 5 shared
// loads and 5 stores instead of 20 more global loads.  One barrier per row.  Same units, same order of the sums per
// thread as observables_kernel.
constexpr int OBS_RING = 4;
template <typename T> struct ObsRing {
    typename vec2<T>::type ring[OBS_RING][10][129];   // [slot][plane][column; 128 = the +x neighbour of the last column]
    double2 psi[2][5][129];                            // psi of a row, [row parity][level][column]
};

template <typename T>
__device__ __forceinline__ void obs_cp_async(typename vec2<T>::type* sm, const typename vec2<T>::type* g) {
    if constexpr (sizeof(T) == 8)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(sm)), "l"(g) : "memory");
    else
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(sm)), "l"(g) : "memory");
}

template <typename T>
__global__ void __launch_bounds__(128, sizeof(T) == 8 ? 2 : 3) observables_ring_kernel(const typename vec2<T>::type* __restrict__ q,
                                                          const typename vec2<T>::type* __restrict__ qprev,
                                                          const __grid_constant__ ObsGeom G, double* partials) {
    using V = typename vec2<T>::type;
    extern __shared__ __align__(16) unsigned char obs_smem[];
    ObsRing<T>& S = *reinterpret_cast<ObsRing<T>*>(obs_smem);
    const int64_t n = G.nx * G.ny;
    const int t = threadIdx.x;
    double acc[OBS_NACC];
#pragma unroll
    for (int k = 0; k < OBS_NACC; ++k) acc[k] = 0.0;
    double zr[5] = {0, 0, 0, 0, 0}, zi[5] = {0, 0, 0, 0, 0};        // no z direction in 2D

    const int64_t units = G.ncb * G.nsg;
    for (int64_t u = blockIdx.x; u < units; u += gridDim.x) {
        const int64_t cb = u % G.ncb, sg = u / G.ncb;
        const int64_t xb = G.x0 + cb * 128;
        const int ncols = (int)((G.x1 - xb < 128) ? G.x1 - xb : 128);
        const bool own = t < ncols;                                     // this thread sums a column
        const int64_t x = xb + (own ? t : 0);
        const int64_t xe = (xb + ncols == G.nx) ? 0 : xb + ncols;       // the +x neighbour of the unit's last column
        const int64_t ys = G.y0 + sg * G.seg;
        const int64_t ye = (ys + G.seg < G.y1) ? ys + G.seg : G.y1;
        const int nr = (int)(ye - ys);                                  // rows summed; rows ys .. ye are needed
        // copy row ys + i (periodic) of this thread's column (thread 0: also of column xe) into slot i mod R
        auto issue = [&](int i) {
            if (i <= nr) {
                int64_t y = ys + i;
                if (y >= G.ny) y -= G.ny;
                const V* g = q + y * G.nx;
                V (*slot)[129] = S.ring[i % OBS_RING];
                if (own) {
#pragma unroll
                    for (int pl = 0; pl < 10; ++pl) obs_cp_async<T>(&slot[pl][t], g + (int64_t)pl * n + x);
                }
                if (t == 0) {
#pragma unroll
                    for (int pl = 0; pl < 10; ++pl) obs_cp_async<T>(&slot[pl][ncols], g + (int64_t)pl * n + xe);
                }
            }
            asm volatile("cp.async.commit_group;" ::: "memory");
        };
        // psi and |q|^2 of column c of the row in `slot`
        auto form = [&](int slot, int c, double pr[5], double pi[5], double& nq) {
            nq = 0.0;
#pragma unroll
            for (int j = 0; j < 5; ++j) {
                const V a = S.ring[slot][2 * j][c], b = S.ring[slot][2 * j + 1][c];
                const double ar = a.x, ai = a.y, br = b.x, bi = b.y;
                pr[j] = ar + br; pi[j] = ai + bi;
                nq += ar * ar + ai * ai + br * br + bi * bi;
            }
        };
        auto publish = [&](int par, int c, const double pr[5], const double pi[5]) {
#pragma unroll
            for (int j = 0; j < 5; ++j) S.psi[par][j][c] = make_double2(pr[j], pi[j]);
        };

        __syncthreads();                                   // the previous unit's readers are done with the ring
#pragma unroll
        for (int i = 0; i < OBS_RING - 1; ++i) issue(i);
        asm volatile("cp.async.wait_group %0;" ::"n"(OBS_RING - 2) : "memory");      // row ys has landed
        __syncthreads();
        double pr[5], pi[5], nq = 0.0;
        if (own) { form(0, t, pr, pi, nq); publish(0, t, pr, pi); }
        if (t == 0) { double er[5], ei[5], en; form(0, ncols, er, ei, en); publish(0, ncols, er, ei); }
        for (int i = 0; i < nr; ++i) {
            asm volatile("cp.async.wait_group %0;" ::"n"(OBS_RING - 3) : "memory");  // row ys + i + 1 has landed
            __syncthreads();                               // ... for every thread; psi of row ys + i is published
            issue(i + OBS_RING - 1);                       // into the slot of row ys + i - 1
            double yr[5], yi[5], ynq = 0.0, xr[5], xi[5], or_[5], oi[5];
            if (own) {
                form((i + 1) % OBS_RING, t, yr, yi, ynq);
                publish((i + 1) & 1, t, yr, yi);
            }
            if (t == 0) { double er[5], ei[5], en; form((i + 1) % OBS_RING, ncols, er, ei, en); publish((i + 1) & 1, ncols, er, ei); }
            if (own) {
#pragma unroll
                for (int j = 0; j < 5; ++j) { const double2 v = S.psi[i & 1][j][t + 1]; xr[j] = v.x; xi[j] = v.y; }
                if (qprev) load_psi<T>(qprev, n, (ys + i) * G.nx + x, or_, oi, nullptr);
                obs_site(acc, 2, qprev != nullptr, nq, pr, pi, xr, xi, yr, yi, zr, zi, or_, oi);
#pragma unroll
                for (int j = 0; j < 5; ++j) { pr[j] = yr[j]; pi[j] = yi[j]; }
                nq = ynq;
            }
        }
        asm volatile("cp.async.wait_group 0;" ::: "memory");
    }

    __shared__ double sm[4][OBS_NACC];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < OBS_NACC; ++k) {
        double v = acc[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) sm[warp][k] = v;
    }
    __syncthreads();
    if (threadIdx.x < OBS_NACC) {
        double v = 0.0;
        for (int w = 0; w < 4; ++w) v += sm[w][threadIdx.x];
        partials[(int64_t)blockIdx.x * OBS_NACC + threadIdx.x] = v;
    }
}

__global__ void __launch_bounds__(256) reduce_partials_kernel(const double* partials, int nblocks,
                                                              double* sums) {
    __shared__ double sm[8];
    for (int k = 0; k < OBS_NACC; ++k) {
        double v = 0.0;
        for (int b = threadIdx.x; b < nblocks; b += blockDim.x) v += partials[(int64_t)b * OBS_NACC + k];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
        __syncthreads();
        if (threadIdx.x == 0) {
            double s = 0.0;
            for (int w = 0; w < 8; ++w) s += sm[w];
            sums[k] = s;
        }
        __syncthreads();
    }
}

cudaError_t launch_observables(const Launch& L, qlga_prec prec, const void* q, const void* qprev,
                               int64_t nx, int64_t ny, int64_t nz, int ndim, int64_t r0, int64_t r1,
                               double* partials, int nblocks, double* sums) {
    // r0 .. r1: whole layers of the slowest axis (the owned layers of a slab, else the whole lattice)
    ObsGeom G;
    G.nx = nx; G.ny = ny; G.nz = nz; G.ndim = ndim;
    G.x0 = 0; G.x1 = nx; G.y0 = 0; G.y1 = ny; G.z0 = 0; G.z1 = nz;
    const int64_t layer = (ndim == 1) ? 1 : (ndim == 2 ? nx : nx * ny);
    if (r0 % layer != 0 || r1 % layer != 0 || r1 <= r0) return cudaErrorInvalidValue;
    if (ndim == 1) { G.x0 = r0; G.x1 = r1; } else if (ndim == 2) { G.y0 = r0 / layer; G.y1 = r1 / layer; }
    else { G.z0 = r0 / layer; G.z1 = r1 / layer; }
    G.ncb = (G.x1 - G.x0 + 127) / 128;
    // segments: about four units per block, at least 16 rows each (the first row of a unit is loaded twice)
    const int64_t rows = G.y1 - G.y0;
    int64_t nsg = (4 * (int64_t)nblocks + G.ncb * (G.z1 - G.z0) - 1) / (G.ncb * (G.z1 - G.z0));
    if (nsg > rows / 16) nsg = rows / 16;
    if (nsg < 1) nsg = 1;
    G.seg = (rows + nsg - 1) / nsg;
    G.nsg = (rows + G.seg - 1) / G.seg;
    const int64_t units = G.ncb * G.nsg * (G.z1 - G.z0);
    if (units < nblocks) nblocks = (int)units;
    if (ndim == 2) {
        // (the shared-memory opt-in is a per-device attribute of the function: set on every launch, idempotent and cheap)
        cudaError_t e;
        if (prec == QLGA_F64) {
            e = cudaFuncSetAttribute(observables_ring_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(ObsRing<double>));
            if (e != cudaSuccess) return e;
            observables_ring_kernel<double><<<nblocks, 128, sizeof(ObsRing<double>), L.stream>>>((const double2*)q, (const double2*)qprev, G, partials);
        } else {
            e = cudaFuncSetAttribute(observables_ring_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(ObsRing<float>));
            if (e != cudaSuccess) return e;
            observables_ring_kernel<float><<<nblocks, 128, sizeof(ObsRing<float>), L.stream>>>((const float2*)q, (const float2*)qprev, G, partials);
        }
    } else if (prec == QLGA_F64)
        observables_kernel<double><<<nblocks, 128, 0, L.stream>>>((const double2*)q, (const double2*)qprev, G, partials);
    else
        observables_kernel<float><<<nblocks, 128, 0, L.stream>>>((const float2*)q, (const float2*)qprev, G, partials);
    ++*L.counter;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    reduce_partials_kernel<<<1, 256, 0, L.stream>>>(partials, nblocks, sums);
    ++*L.counter;
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------
// Lattice vorticity (eq. 102-104, reading R8).  Substituting v_x, v_y into the
// curl, omega(x,y) depends only on psi at the four diagonal neighbours:
//   omega = (1/4)[ arg(p(x+1,y+1) p*(x+1,y-1)) - arg(p(x-1,y+1) p*(x-1,y-1))
//                - arg(p(x+1,y+1) p*(x-1,y+1)) + arg(p(x+1,y-1) p*(x-1,y-1)) ],  arg(0) := 0.
// The arithmetic is done in fp64 for both storage types.
// ---------------------------------------------------------------------------
__device__ __forceinline__ double arg_prod_conj(double ar, double ai, double br, double bi) {
    // arg(a * conj(b)); products rounded one by one (no FMA contraction): the sign of an exactly
    // cancelling imaginary part decides between +pi and -pi
    const double re = __dadd_rn(__dmul_rn(ar, br), __dmul_rn(ai, bi));
    const double im = __dsub_rn(__dmul_rn(ai, br), __dmul_rn(ar, bi));
    return (re == 0.0 && im == 0.0) ? 0.0 : atan2(im, re);
}

// Winding number of the closed loop z0 -> z1 -> z2 -> z3 -> z0 whose edges are the wrapped phase
// differences arg(z_{k+1} conj z_k) in (-pi, pi]: their sum is 2 pi w exactly, so w needs no atan2.
// Each vertex is assigned the quadrant it lies in (half-open, so that the four sectors tile the plane
// without the origin); an edge changes the quadrant count by 0, +-1 (neighbouring quadrants: the short
// arc) or +-2 (opposite quadrants: the sign of Im(z_{k+1} conj z_k) gives the sense of rotation), and
// w = (sum of the changes) / 4.  Returns false in the cases where a wrapped difference is not defined
// by the geometry alone -- a vertex that is exactly zero (arg(0) := 0 breaks the loop) or two opposite
// vertices exactly antiparallel (arg = +-pi by the sign of a zero) -- which take the atan2 path.
__device__ __forceinline__ int quadrant(double re, double im) {
    return (re > 0.0 && im >= 0.0) ? 0 : ((re <= 0.0 && im > 0.0) ? 1 : ((re < 0.0 && im <= 0.0) ? 2 : 3));
}
__device__ __forceinline__ bool loop_winding(const double zr[4], const double zi[4], int* w) {
    int q[4];
    bool ok = true;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        ok = ok && !(zr[k] == 0.0 && zi[k] == 0.0);
        q[k] = quadrant(zr[k], zi[k]);
    }
    int sum = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int t = (k + 1) & 3;
        const int dq = (q[t] - q[k]) & 3;
        // Im(z_t conj z_k), products rounded one by one so that exactly antiparallel vertices give exactly 0
        const double im = __dsub_rn(__dmul_rn(zi[t], zr[k]), __dmul_rn(zr[t], zi[k]));
        ok = ok && !(dq == 2 && im == 0.0);
        sum += (dq == 0) ? 0 : ((dq == 1) ? 1 : ((dq == 3) ? -1 : (im > 0.0 ? 2 : -2)));
    }
    *w = sum / 4;
    return ok;
}

// Tiled (round 2): a CTA of 32 x 8 threads forms psi = q1 + q2 of its (32 + 2) x (8 + 2) sites once, in shared memory
// (every amplitude is read once per tile; the halo, a third of the tile, comes out of L2 where the neighbouring tile's
// CTA has just put it), and every thread takes the winding of its site from the four diagonal neighbours there.  The
// round-1 kernel (one thread per site, every amplitude read four times through L1 / L2) reached 62 % of the copy
// bandwidth.  (Measured and rejected: a column-marching version with a cp.async ring like observables_ring_kernel --
// two CTAs per SM by its 104 KB of shared memory leave eight warps for the branchy winding count: 5.5 ms against 3.3.)
template <typename T>
__global__ void __launch_bounds__(256) vorticity_tile_kernel(const typename vec2<T>::type* __restrict__ q, T* __restrict__ omega,
                                                              int64_t nx, int64_t ny) {
    using V = typename vec2<T>::type;
    __shared__ double2 P[5][10][34];
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * 32 + tx;
    const int64_t xb = (int64_t)blockIdx.x * 32, yb = (int64_t)blockIdx.y * 8, n = nx * ny;
    for (int s = tid; s < 340; s += 256) {
        const int cy = s / 34, cx = s - cy * 34;
        int64_t x = (xb + cx - 1) % nx, y = (yb + cy - 1) % ny;
        if (x < 0) x += nx;
        if (y < 0) y += ny;
        const V* g = q + y * nx + x;
#pragma unroll
        for (int j = 0; j < 5; ++j) {
            const V a = g[(int64_t)(2 * j) * n], b = g[(int64_t)(2 * j + 1) * n];
            P[j][cy][cx] = make_double2((double)a.x + (double)b.x, (double)a.y + (double)b.y);
        }
    }
    __syncthreads();
    const int64_t x = xb + tx, y = yb + ty;
    if (x >= nx || y >= ny) return;
    const int64_t r = y * nx + x;
#pragma unroll
    for (int j = 0; j < 5; ++j) {
        const double2 pp = P[j][ty + 2][tx + 2], pm = P[j][ty][tx + 2];          // (x+1, y+1), (x+1, y-1)
        const double2 mp = P[j][ty + 2][tx], mm = P[j][ty][tx];                  // (x-1, y+1), (x-1, y-1)
        // The four terms are the wrapped phase differences around the closed loop
        // (x+1,y-1) -> (x+1,y+1) -> (x-1,y+1) -> (x-1,y-1) -> (x+1,y-1): omega = (pi/2) x its winding number.
        const double zr[4] = {pm.x, pp.x, mp.x, mm.x}, zi[4] = {pm.y, pp.y, mp.y, mm.y};
        int w;
        if (loop_winding(zr, zi, &w)) {
            omega[(int64_t)j * n + r] = (T)(1.5707963267948966192313216916398 * (double)w);
            continue;
        }
        // degenerate site (a zero or an exactly antiparallel pair among the four): the definition term by term
        // v_y(x+1,y), v_y(x-1,y), v_x(x,y+1), v_x(x,y-1)   (each is half the wrapped phase difference)
        const double vy_p = 0.5 * arg_prod_conj(pp.x, pp.y, pm.x, pm.y);
        const double vy_m = 0.5 * arg_prod_conj(mp.x, mp.y, mm.x, mm.y);
        const double vx_p = 0.5 * arg_prod_conj(pp.x, pp.y, mp.x, mp.y);
        const double vx_m = 0.5 * arg_prod_conj(pm.x, pm.y, mm.x, mm.y);
        omega[(int64_t)j * n + r] = (T)(0.5 * (vy_p - vy_m - vx_p + vx_m));
    }
}

cudaError_t launch_vorticity(const Launch& L, qlga_prec prec, const void* q, void* omega,
                             int64_t nx, int64_t ny) {
    const int64_t bx = (nx + 31) / 32, by = (ny + 7) / 8;
    if (bx > 2147483647LL || by > 65535) return cudaErrorInvalidValue;
    const dim3 grid((unsigned)bx, (unsigned)by), block(32, 8);
    if (prec == QLGA_F64)
        vorticity_tile_kernel<double><<<grid, block, 0, L.stream>>>((const double2*)q, (double*)omega, nx, ny);
    else
        vorticity_tile_kernel<float><<<grid, block, 0, L.stream>>>((const float2*)q, (float*)omega, nx, ny);
    ++*L.counter;
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------
// psi <-> q.  `psi` points at a chunk holding sites [offset, offset+count) of all
// five channels, packed as [5][count]; q is the full [5][2][nsites] state.
// ---------------------------------------------------------------------------
template <typename T>
__global__ void split_psi_kernel(const typename vec2<T>::type* psi, typename vec2<T>::type* q,
                                 int64_t nsites, int64_t offset, int64_t count) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= 5 * count) return;
    const int64_t j = k / count, r = k % count;
    typename vec2<T>::type v = psi[k];
    v.x *= (T)0.5; v.y *= (T)0.5;                 // q1 = q2 = psi/2  (reading R6)
    q[(2 * j) * nsites + offset + r] = v;
    q[(2 * j + 1) * nsites + offset + r] = v;
}

template <typename T>
__global__ void sum_psi_kernel(const typename vec2<T>::type* q, typename vec2<T>::type* psi,
                               int64_t nsites, int64_t offset, int64_t count) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= 5 * count) return;
    const int64_t j = k / count, r = k % count;
    const typename vec2<T>::type a = q[(2 * j) * nsites + offset + r], b = q[(2 * j + 1) * nsites + offset + r];
    typename vec2<T>::type v; v.x = a.x + b.x; v.y = a.y + b.y;
    psi[k] = v;
}

cudaError_t launch_split_psi(const Launch& L, qlga_prec prec, const void* psi, void* q,
                             int64_t nsites, int64_t offset, int64_t count) {
    const unsigned blocks = (unsigned)((5 * count + 255) / 256);
    if (prec == QLGA_F64)
        split_psi_kernel<double><<<blocks, 256, 0, L.stream>>>((const double2*)psi, (double2*)q, nsites, offset, count);
    else
        split_psi_kernel<float><<<blocks, 256, 0, L.stream>>>((const float2*)psi, (float2*)q, nsites, offset, count);
    ++*L.counter;
    return cudaGetLastError();
}

cudaError_t launch_sum_psi(const Launch& L, qlga_prec prec, const void* q, void* psi,
                           int64_t nsites, int64_t offset, int64_t count) {
    const unsigned blocks = (unsigned)((5 * count + 255) / 256);
    if (prec == QLGA_F64)
        sum_psi_kernel<double><<<blocks, 256, 0, L.stream>>>((const double2*)q, (double2*)psi, nsites, offset, count);
    else
        sum_psi_kernel<float><<<blocks, 256, 0, L.stream>>>((const float2*)q, (float2*)psi, nsites, offset, count);
    ++*L.counter;
    return cudaGetLastError();
}

}  // namespace qlga

// ---------------------------------------------------------------------------
// Total density, the L2 error of eq. (115) and plaquette winding numbers
// (definitions in include/qlga.h).
// ---------------------------------------------------------------------------
namespace qlga {

template <typename T>
__device__ __forceinline__ double site_density(const typename vec2<T>::type* q, int64_t n, int64_t r) {
    double s = 0.0;
#pragma unroll
    for (int j = 0; j < 5; ++j) {
        const typename vec2<T>::type a = q[(int64_t)(2 * j) * n + r], b = q[(int64_t)(2 * j + 1) * n + r];
        const double pr = (double)a.x + (double)b.x, pi = (double)a.y + (double)b.y;
        s += pr * pr + pi * pi;
    }
    return s;
}

template <typename T>
__global__ void density_kernel(const typename vec2<T>::type* q, T* rho, int64_t n) {
    const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r < n) rho[r] = (T)site_density<T>(q, n, r);
}

template <typename T>
__global__ void __launch_bounds__(256) l2_error_kernel(const typename vec2<T>::type* q, const T* rho_ref,
                                                       int64_t n, double* partials) {
    double acc = 0.0;
    for (int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; r < n; r += (int64_t)gridDim.x * blockDim.x) {
        const double d = (double)rho_ref[r] - site_density<T>(q, n, r);
        acc += d * d;
    }
    __shared__ double sm[8];
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < 8; ++w) s += sm[w];
        partials[(int64_t)blockIdx.x * OBS_NACC] = s;
        for (int k = 1; k < OBS_NACC; ++k) partials[(int64_t)blockIdx.x * OBS_NACC + k] = 0.0;
    }
}

template <typename T>
__global__ void __launch_bounds__(128) vortices_kernel(const typename vec2<T>::type* q, int64_t nx, int64_t ny,
                                                       int* list, long long max_out, unsigned long long* counter) {
    using V = typename vec2<T>::type;
    const int64_t n = nx * ny;
    const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n) return;
    const int64_t x = r % nx, y = r / nx;
    const int64_t xp = (x == nx - 1) ? 0 : x + 1, yp = (y == ny - 1) ? 0 : y + 1;
    const int64_t ia = r, ib = y * nx + xp, ic = yp * nx + xp, id = yp * nx + x;
    for (int j = 0; j < 5; ++j) {
        const V* p1 = q + (int64_t)(2 * j) * n;
        const V* p2 = q + (int64_t)(2 * j + 1) * n;
        V u, v;
        u = p1[ia]; v = p2[ia]; const double ar = (double)u.x + (double)v.x, ai = (double)u.y + (double)v.y;
        u = p1[ib]; v = p2[ib]; const double br = (double)u.x + (double)v.x, bi = (double)u.y + (double)v.y;
        u = p1[ic]; v = p2[ic]; const double cr = (double)u.x + (double)v.x, ci = (double)u.y + (double)v.y;
        u = p1[id]; v = p2[id]; const double dr = (double)u.x + (double)v.x, di = (double)u.y + (double)v.y;
        const double zr[4] = {ar, br, cr, dr}, zi[4] = {ai, bi, ci, di};
        int w;
        if (!loop_winding(zr, zi, &w)) {          // degenerate plaquette: the definition term by term
            const double circ = arg_prod_conj(br, bi, ar, ai) + arg_prod_conj(cr, ci, br, bi)
                              + arg_prod_conj(dr, di, cr, ci) + arg_prod_conj(ar, ai, dr, di);
            w = (int)rint(circ * 0.15915494309189533576888376337251);            // 1/(2 pi)
        }
        if (w != 0) {
            const unsigned long long slot = atomicAdd(counter, 1ULL);
            if ((long long)slot < max_out) {
                int4 rec; rec.x = j; rec.y = (int)x; rec.z = (int)y; rec.w = w;
                reinterpret_cast<int4*>(list)[slot] = rec;
            }
        }
    }
}

cudaError_t launch_density(const Launch& L, qlga_prec prec, const void* q, void* rho, int64_t n) {
    const unsigned blocks = (unsigned)((n + 255) / 256);
    if (prec == QLGA_F64) density_kernel<double><<<blocks, 256, 0, L.stream>>>((const double2*)q, (double*)rho, n);
    else density_kernel<float><<<blocks, 256, 0, L.stream>>>((const float2*)q, (float*)rho, n);
    ++*L.counter;
    return cudaGetLastError();
}

cudaError_t launch_l2_error(const Launch& L, qlga_prec prec, const void* q, const void* rho_ref, int64_t n,
                            double* partials, int nblocks, double* sums) {
    if (prec == QLGA_F64)
        l2_error_kernel<double><<<nblocks, 256, 0, L.stream>>>((const double2*)q, (const double*)rho_ref, n, partials);
    else
        l2_error_kernel<float><<<nblocks, 256, 0, L.stream>>>((const float2*)q, (const float*)rho_ref, n, partials);
    ++*L.counter;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    reduce_partials_kernel<<<1, 256, 0, L.stream>>>(partials, nblocks, sums);
    ++*L.counter;
    return cudaGetLastError();
}

cudaError_t launch_vortices(const Launch& L, qlga_prec prec, const void* q, int64_t nx, int64_t ny,
                            int* list, long long max_out, unsigned long long* counter) {
    const int64_t n = nx * ny;
    const unsigned blocks = (unsigned)((n + 127) / 128);
    if (prec == QLGA_F64)
        vortices_kernel<double><<<blocks, 128, 0, L.stream>>>((const double2*)q, nx, ny, list, max_out, counter);
    else
        vortices_kernel<float><<<blocks, 128, 0, L.stream>>>((const float2*)q, nx, ny, list, max_out, counter);
    ++*L.counter;
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------
// Interaction-angle statistics (qlga_angle_stats): per site the angle bound the pass kernels select
// the polynomial degree by, theta = s (2|c1||F| + |c2| rho / 5), and the scalar phase s (c0 rho + mu).
// out: [0] double sum theta, [1] uint bits of max theta | uint bits of max |phase|, [2..14] degree histogram.
// ---------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) angle_stats_kernel(const typename vec2<T>::type* q, int64_t n,
                                                          double tg1, double tg2, double g0, double smu,
                                                          const __grid_constant__ ExpTable tab,
                                                          unsigned long long* out) {
    __shared__ unsigned int sh_hist[13];
    __shared__ unsigned int sh_max[2];
    __shared__ double sh_sum[8];
    if (threadIdx.x < 13) sh_hist[threadIdx.x] = 0;
    if (threadIdx.x < 2) sh_max[threadIdx.x] = 0;
    __syncthreads();
    double sum = 0.0;
    float tmax = 0.f, pmax = 0.f;
    const double rt6 = 2.4494897427831780981972840747059;
    for (int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; r < n; r += (int64_t)gridDim.x * blockDim.x) {
        double pr[5], pi[5], nm[5];
        load_psi<T>(q, n, r, pr, pi, nullptr);
#pragma unroll
        for (int j = 0; j < 5; ++j) nm[j] = pr[j] * pr[j] + pi[j] * pi[j];
        const double rho = nm[0] + nm[1] + nm[2] + nm[3] + nm[4];
        const double Fz = 2.0 * (nm[0] - nm[4]) + (nm[1] - nm[3]);
        const double far_ = pr[0] * pr[1] + pi[0] * pi[1] + pr[3] * pr[4] + pi[3] * pi[4];
        const double fai = pr[0] * pi[1] - pi[0] * pr[1] + pr[3] * pi[4] - pi[3] * pr[4];
        const double fbr = pr[1] * pr[2] + pi[1] * pi[2] + pr[2] * pr[3] + pi[2] * pi[3];
        const double fbi = pr[1] * pi[2] - pi[1] * pr[2] + pr[2] * pi[3] - pi[2] * pr[3];
        const double Fx = 2.0 * far_ + rt6 * fbr, Fy = 2.0 * fai + rt6 * fbi;
        const double theta = tg1 * sqrt(Fx * Fx + Fy * Fy + Fz * Fz) + tg2 * rho;
        const float th = (float)theta;
        sum += theta;
        tmax = fmaxf(tmax, th);
        pmax = fmaxf(pmax, (float)fabs(g0 * rho + smu));
        int p = 0;
        if (th <= tab.theta_split) p = lut_degree(tab, th * 1.0009765625f);
        atomicAdd(&sh_hist[p], 1u);
    }
    atomicMax(&sh_max[0], __float_as_uint(tmax));
    atomicMax(&sh_max[1], __float_as_uint(pmax));
    for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
    if ((threadIdx.x & 31) == 0) sh_sum[threadIdx.x >> 5] = sum;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < 8; ++w) s += sh_sum[w];
        atomicAdd(reinterpret_cast<double*>(out), s);
        atomicMax(reinterpret_cast<unsigned int*>(out + 1), sh_max[0]);
        atomicMax(reinterpret_cast<unsigned int*>(out + 1) + 1, sh_max[1]);
    }
    if (threadIdx.x < 13 && sh_hist[threadIdx.x]) atomicAdd(out + 2 + threadIdx.x, (unsigned long long)sh_hist[threadIdx.x]);
}

cudaError_t launch_angle_stats(const Launch& L, qlga_prec prec, const void* q, int64_t n, double tg1, double tg2,
                               double g0, double smu, const ExpTable& tab, int nblocks, unsigned long long* out) {
    if (prec == QLGA_F64)
        angle_stats_kernel<double><<<nblocks, 256, 0, L.stream>>>((const double2*)q, n, tg1, tg2, g0, smu, tab, out);
    else
        angle_stats_kernel<float><<<nblocks, 256, 0, L.stream>>>((const float2*)q, n, tg1, tg2, g0, smu, tab, out);
    ++*L.counter;
    return cudaGetLastError();
}

}  // namespace qlga

// ---------------------------------------------------------------------------
// qlga_observable_sums_noalloc (include/qlga.h): the observables reduction for callers that cannot call
// cudaMalloc (CUDA graph capture, serving loops, harnesses that forbid it).  It needs no context and
// allocates nothing: the per-block partial sums and the 19 reduced sums live in the file-scope device
// array below, QLGA_NOALLOC_MAX_BLOCKS x 19 + 19 doubles = 311 448 bytes that every GPU loading the
// library holds until exit.  Same kernels as qlga_observable_sums (observables_kernel,
// reduce_partials_kernel), same grid: bit-identical sums.
//
// In host code the name `g_noalloc_scratch` is a host-side stand-in, not a device address: the address is
// taken once per device, with that device current, by cudaGetSymbolAddress, and that pointer goes to the
// kernels.  Every call shares the array: nothing in it has to start at zero (each block overwrites all 19
// of its partials and the second pass reads exactly the blocks just written), but two calls that overlap
// on the GPU (different streams, no ordering between them) race on it.
// ---------------------------------------------------------------------------
namespace qlga {
constexpr int NOALLOC_DOUBLES = QLGA_NOALLOC_MAX_BLOCKS * OBS_NACC + OBS_NACC;
static __device__ __align__(256) double g_noalloc_scratch[NOALLOC_DOUBLES];
}  // namespace qlga

#include <atomic>
#include <stdio.h>

static char g_noalloc_err[256] = "";
extern "C" const char* qlga_noalloc_last_error(void) { return g_noalloc_err; }

static qlga_status noalloc_fail(qlga_status st, const char* text, cudaError_t e = cudaSuccess) {
    if (e != cudaSuccess) snprintf(g_noalloc_err, sizeof(g_noalloc_err), "%s: %s", text, cudaGetErrorString(e));
    else snprintf(g_noalloc_err, sizeof(g_noalloc_err), "%s", text);
    return st;
}

extern "C" qlga_status qlga_observable_sums_noalloc(const void* dev_q, const void* dev_qprev, int ndim,
                                                    const int64_t* dims, qlga_prec prec, int nblocks,
                                                    double* dev_sums, void* cuda_stream) {
    using namespace qlga;
    if (!dev_q || !dev_sums || !dims || ndim < 1 || ndim > 3)
        return noalloc_fail(QLGA_EINVAL, "qlga_observable_sums_noalloc: NULL pointer or bad ndim");
    const int64_t nx = dims[0], ny = dims[1], nz = (ndim == 3) ? dims[2] : 1;
    if (nx < 1 || ny < 1 || nz < 1 || (ndim == 1 && ny != 1) || (double)nx * (double)ny * (double)nz > 1.0e12)
        return noalloc_fail(QLGA_EINVAL, "qlga_observable_sums_noalloc: bad dims");
    if (prec != QLGA_F64 && prec != QLGA_F32 && prec != QLGA_F32X)
        return noalloc_fail(QLGA_EINVAL, "qlga_observable_sums_noalloc: bad precision");
    if (nblocks < 0 || nblocks > QLGA_NOALLOC_MAX_BLOCKS)
        return noalloc_fail(QLGA_EINVAL, "qlga_observable_sums_noalloc: nblocks beyond QLGA_NOALLOC_MAX_BLOCKS (2048): "
                                         "the static scratch holds 19 partial sums for at most that many blocks");
    // the device that holds the state; run there whatever device is current, restore on return
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, dev_q);
    if (e != cudaSuccess) { cudaGetLastError(); return noalloc_fail(QLGA_ECUDA, "qlga_observable_sums_noalloc: cudaPointerGetAttributes", e); }
    if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)
        return noalloc_fail(QLGA_EINVAL, "qlga_observable_sums_noalloc: dev_q is not device memory");
    const int dev = at.device;
    if (dev < 0 || dev >= 64) return noalloc_fail(QLGA_EUNSUP, "qlga_observable_sums_noalloc: device ordinal beyond 63");
    int caller_dev = -1;
    if ((e = cudaGetDevice(&caller_dev)) != cudaSuccess) return noalloc_fail(QLGA_ECUDA, "cudaGetDevice", e);
    const bool switched = caller_dev != dev;
    if (switched && (e = cudaSetDevice(dev)) != cudaSuccess) return noalloc_fail(QLGA_ECUDA, "cudaSetDevice", e);

    // set-up, once per device, with that device current: the device address of the static array and the SM count
    static std::atomic<double*> scratch_of[64];
    static std::atomic<int> sms_of[64];
    qlga_status st = QLGA_OK;
    double* scratch = scratch_of[dev].load(std::memory_order_acquire);
    if (!scratch) {
        double* p = nullptr;
        int sms = 0;
        e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            st = noalloc_fail(QLGA_ECUDA, "qlga_observable_sums_noalloc: cudaGetSymbolAddress(static scratch)", e);
        } else {
            sms_of[dev].store(sms, std::memory_order_relaxed);
            scratch_of[dev].store(p, std::memory_order_release);
            scratch = p;
        }
    }
    if (st == QLGA_OK) {
        const int64_t n = nx * ny * nz;
        int blocks = nblocks ? nblocks : sms_of[dev].load(std::memory_order_relaxed) * 8;     // qlga_observable_sums' grid
        if (blocks > QLGA_NOALLOC_MAX_BLOCKS) blocks = QLGA_NOALLOC_MAX_BLOCKS;
        if ((int64_t)blocks * 256 > n) blocks = (int)((n + 255) / 256);
        int64_t launches = 0;
        Launch L{(cudaStream_t)cuda_stream, &launches, dev};
        double* partials = scratch;
        double* sums = scratch + (size_t)QLGA_NOALLOC_MAX_BLOCKS * OBS_NACC;
        e = launch_observables(L, prec == QLGA_F64 ? QLGA_F64 : QLGA_F32, dev_q, dev_qprev, nx, ny, nz, ndim, 0, n,
                               partials, blocks, sums);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(dev_sums, sums, sizeof(double) * QLGA_NSUMS, cudaMemcpyDeviceToDevice, L.stream);
        if (e != cudaSuccess) { cudaGetLastError(); st = noalloc_fail(QLGA_ECUDA, "qlga_observable_sums_noalloc: launch", e); }
    }
    if (switched) cudaSetDevice(caller_dev);
    return st;
}
