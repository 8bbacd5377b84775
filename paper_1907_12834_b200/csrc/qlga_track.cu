// qlga_track.cu -- association of two vortex detections (the tracking half;
// the paper follows "vortices with a positive / negative winding number" as red / blue tracks, Figs. 18, 21,
// 22, without printing the tracker; reading R18 of DESIGN.md).
//
// A detection is a list of records (j, x, y, w) of qlga_vortices.  Two records can be the same vortex at two
// times only if they agree in channel j and winding w.  Distance: the periodic (minimal-image) squared
// lattice distance d2 = dx^2 + dy^2, an integer.  The nearest candidate of a record is the one that minimises
// (d2, y, x) lexicographically (the tie-break makes it independent of the order of the lists) among the
// records of the other list with the same (j, w) and d2 <= max_d2.  Two records are matched iff each is the
// other's nearest candidate (mutual nearest neighbours).  Integer work throughout: bit-exact against the oracle.
#include "qlga_internal.h"

namespace qlga {

__device__ __forceinline__ long long wrap_d2(int4 a, int4 b, int nx, int ny) {
    int dx = abs(a.y - b.y), dy = abs(a.z - b.z);
    dx = min(dx, nx - dx);
    dy = min(dy, ny - dy);
    return (long long)dx * dx + (long long)dy * dy;
}

// nn[i] = index in b of the nearest candidate of a[i], or -1
__global__ void __launch_bounds__(128) nearest_kernel(const int4* __restrict__ a, int na, const int4* __restrict__ b, int nb,
                                                      int nx, int ny, long long max_d2, int* __restrict__ nn) {
    __shared__ int4 tile[128];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int4 me = (i < na) ? a[i] : make_int4(-1, 0, 0, 0);
    long long best = -1;
    int best_k = -1, best_y = 0, best_x = 0;
    for (int base = 0; base < nb; base += 128) {
        const int k = base + threadIdx.x;
        tile[threadIdx.x] = (k < nb) ? b[k] : make_int4(-2, 0, 0, 0);
        __syncthreads();
        const int lim = min(128, nb - base);
        for (int t = 0; t < lim; ++t) {
            const int4 c = tile[t];
            if (c.x != me.x || c.w != me.w) continue;
            const long long d2 = wrap_d2(me, c, nx, ny);
            if (d2 > max_d2) continue;
            const bool better = best_k < 0 || d2 < best || (d2 == best && (c.z < best_y || (c.z == best_y && c.y < best_x)));
            if (better) { best = d2; best_k = base + t; best_y = c.z; best_x = c.y; }
        }
        __syncthreads();
    }
    if (i < na) nn[i] = best_k;
}

// match_a[i] = nn_a[i] if nn_b[nn_a[i]] == i else -1
__global__ void mutual_kernel(const int* __restrict__ nn_a, int na, const int* __restrict__ nn_b, int* __restrict__ match_a) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= na) return;
    const int k = nn_a[i];
    match_a[i] = (k >= 0 && nn_b[k] == i) ? k : -1;
}

cudaError_t launch_vortex_match(const Launch& L, const int* prev, int np, const int* cur, int nc, int nx, int ny,
                                long long max_d2, int* nn_cur, int* nn_prev, int* match_cur, int* match_prev) {
    if (nc > 0) {
        nearest_kernel<<<(nc + 127) / 128, 128, 0, L.stream>>>((const int4*)cur, nc, (const int4*)prev, np, nx, ny, max_d2, nn_cur);
        ++*L.counter;
    }
    if (np > 0) {
        nearest_kernel<<<(np + 127) / 128, 128, 0, L.stream>>>((const int4*)prev, np, (const int4*)cur, nc, nx, ny, max_d2, nn_prev);
        ++*L.counter;
    }
    if (nc > 0) { mutual_kernel<<<(nc + 127) / 128, 128, 0, L.stream>>>(nn_cur, nc, nn_prev, match_cur); ++*L.counter; }
    if (np > 0) { mutual_kernel<<<(np + 127) / 128, 128, 0, L.stream>>>(nn_prev, np, nn_cur, match_prev); ++*L.counter; }
    return cudaGetLastError();
}

}  // namespace qlga
