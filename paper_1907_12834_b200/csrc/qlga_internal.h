// qlga_internal.h -- context and kernel-launcher declarations shared by the
// translation units of libqlga.so.  Not part of the public ABI (include/qlga.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/qlga.h"
#include "qlga_math.cuh"

namespace qlga {

// Parameters of one fused directional pass (4 kinetic factors per fused time
// step, with the interaction interleaved as `umode` says).
struct PassParams {
    const void* src;
    void* dst;
    int64_t nx, ny, nz;    // lattice (ny = nz = 1 in 1D, nz = 1 in 2D)
    int ksteps;            // time steps fused in this launch (1 in 2D)
    int umode;             // 0: no U in this pass, 1: U before the first factor of each step,
                           // 2: U before every factor
    double g[4][3];        // per factor: (s c0, s c1, s c2/5) * 4^-e  (e = deferred halvings so far)
    double smu;            // s * mu, the chemical-potential phase of one U (not scaled: it multiplies no density)
    int utail;             // plain ordering: apply the NEXT step's U (constants gt) after this pass's last factor
    double gt[3];          // (c0, c1, c2/5): the full-angle U on the unscaled state
    double out_scale;      // 2^-4, applied after the 4 factors of a step
    int* flag;             // device error word of the context (FLAG_* in qlga_math.cuh)
    ExpTable tab;
    // Band mode (qlga_band.cu): source and destination are different views of the lattice.  0 = the lattice's own.
    int64_t src_plane = 0; // elements between consecutive planes of src (default nx*ny*nz)
    int64_t dst_plane = 0; // the same for dst
    // marching pass only: output rows [row_begin, row_end) of the line (default the whole line); row r is stored
    // at row r - dst_row_origin of dst (a band buffer that starts at row dst_row_origin of the lattice)
    int64_t row_begin = 0, row_end = 0, dst_row_origin = 0;
#ifdef QLGA_TRACE
    unsigned long long* trace = nullptr; int trace_id = 0;   // debug build: first start / last end (globaltimer) per launch
#endif
};

struct Launch {
    cudaStream_t stream;
    int64_t* counter;      // incremented per kernel launched
    int device;            // the context's device (per-device function attributes)
};

// fused passes (qlga_step.cu); dir = 0 (x), 1 (y) or 2 (z).  `threads` / `cx` are tunables
// (0 = default).  Returns cudaGetLastError().
cudaError_t launch_pass(const Launch& L, qlga_prec prec, int dir, const PassParams& P,
                        int threads, int cx);
// the three instantiation sets (qlga_step.cu, qlga_step_f32.cu, qlga_step_mixed.cu)
cudaError_t launch_pass_f64(const Launch& L, int dir, const PassParams& P, int threads, int cx);
cudaError_t launch_pass_f32(const Launch& L, int dir, const PassParams& P, int threads, int cx);
cudaError_t launch_pass_mixed(const Launch& L, int dir, const PassParams& P, int threads, int cx);
// true if the (columns, threads) pair of a strided pass / the CTA size of the x pass has an instantiation
bool pass_tile_supported(int dir, int threads, int cx);
// interaction-free strided pass by column marching (qlga_march.cu): same arithmetic, no shared memory
bool march_supported(int dir, const PassParams& P);
cudaError_t launch_march(const Launch& L, qlga_prec prec, int dir, const PassParams& P);
// widest ksteps the x pass supports with the given CTA size
int max_ksteps(int threads);

// one kernel per operator (reference path on the GPU)
cudaError_t launch_interaction(const Launch& L, qlga_prec prec, void* q, int64_t nsites,
                               const double g[3], double smu, const ExpTable& tab, int* flag);
cudaError_t launch_kinetic(const Launch& L, qlga_prec prec, const void* src, void* dst,
                           int64_t nx, int64_t ny, int64_t nz, int dir, int sigma);

// diagnostics and state conversion (qlga_diag.cu); `prec` here is the STORAGE precision
// (QLGA_F32X stores fp32: callers pass storage_prec())
constexpr int OBS_NACC = 19;   // accumulators per block, see qlga_diag.cu
cudaError_t launch_observables(const Launch& L, qlga_prec prec, const void* q, const void* qprev,
                               int64_t nx, int64_t ny, int64_t nz, int ndim, int64_t r0, int64_t r1,
                               double* partials, int nblocks, double* sums);
cudaError_t launch_vorticity(const Launch& L, qlga_prec prec, const void* q, void* omega,
                             int64_t nx, int64_t ny);
cudaError_t launch_density(const Launch& L, qlga_prec prec, const void* q, void* rho, int64_t nsites);
cudaError_t launch_l2_error(const Launch& L, qlga_prec prec, const void* q, const void* rho_ref, int64_t nsites,
                            double* partials, int nblocks, double* sums);
cudaError_t launch_vortices(const Launch& L, qlga_prec prec, const void* q, int64_t nx, int64_t ny,
                            int* list, long long max_out, unsigned long long* counter);
cudaError_t launch_angle_stats(const Launch& L, qlga_prec prec, const void* q, int64_t nsites, double tg1, double tg2,
                               double g0, double smu, const ExpTable& tab, int nblocks, unsigned long long* out /*[15]*/);
// association of two vortex detections (qlga_track.cu); all pointers DEVICE, records int32 [n][4] = (j, x, y, w)
cudaError_t launch_vortex_match(const Launch& L, const int* prev, int np, const int* cur, int nc, int nx, int ny,
                                long long max_d2, int* nn_cur, int* nn_prev, int* match_cur, int* match_prev);
cudaError_t launch_split_psi(const Launch& L, qlga_prec prec, const void* psi, void* q,
                             int64_t nsites, int64_t offset, int64_t count);
cudaError_t launch_sum_psi(const Launch& L, qlga_prec prec, const void* q, void* psi,
                           int64_t nsites, int64_t offset, int64_t count);

}  // namespace qlga

struct qlga_ctx {
    int device;            // CUDA device the context (its buffers, stream and scratch) lives on
    int ndim;
    int64_t nx, ny, nz;
    double c[3];
    double mu;             // chemical potential (0 unless qlga_set_chemical_potential)
    qlga_order order;
    qlga_prec prec;
    void* buf[3];
    size_t buf_bytes;
    cudaStream_t stream;
    int cur;               // index of the buffer holding the current state
    int prev;              // index of the buffer holding the previous step's state, or -1
    int have_state;
    int64_t ghost;         // slab decomposition: ghost layers on each side of the slowest axis (0 = none)
    int64_t step;
    int64_t launches;
    // options
    int path;              // 0 fused, 1 per-operator
    int steps_per_launch;  // 1D temporal blocking, 0 = auto
    int fuse_plain_u;      // plain ordering, 2D/3D: the next step's U rides on the x pass (default on)
    int march;             // interaction-free strided passes by column marching (default on; 0 = tile kernel)
    int tol_log2;
    int exp_poly;          // 0 economised, 1 Taylor (QLGA_OPT_EXP_POLY)
    int exp_mod_shift;     // modulus part of the truncation error held to 2^(tol_log2 - shift) (QLGA_OPT_EXP_MOD_SHIFT)
    int f32_phase;         // phase-factor formulation of the fp32 kernels (QLGA_OPT_F32_PHASE)
    int threads_x;
    int tile_y;
    int threads_y;
    int band;              // plain ordering in 2D: one HBM round trip per step by band pipelining (QLGA_OPT_BAND)
    int band_rows;         // rows per band, 0 = auto (QLGA_OPT_BAND_ROWS)
    int band_slots;        // slots of the band ring, 0 = auto (QLGA_OPT_BAND_SLOTS)
    qlga::ExpTable tab;
    // band mode (qlga_api.cu, step_band): the ring that carries the y pass's output to the x pass through L2, the
    // library's own streams (capture origin, y, x0, x1), the events that order the bands, the instantiated graphs
    void* d_band;
    size_t band_bytes;
    cudaStream_t band_stream[4];
    cudaEvent_t* band_ev;
    int band_nev;
    struct BandGraph { int src, dst, tail; int64_t rows, slots; cudaGraphExec_t exec; int64_t nodes; } band_graph[12];
    int band_ngraph;
    // scratch owned by the library
    double* d_partials;    // [obs_blocks][OBS_NACC]
    double* d_sums;        // [OBS_NACC]
    int obs_blocks;
    void* d_stage;         // staging for psi transfers
    size_t stage_bytes;
    void* d_scratch;       // grow-only scratch of the diagnostics with a host destination (density, omega, vortex lists)
    size_t scratch_bytes;
    int* d_flag;           // device error word (FLAG_* in qlga_math.cuh), read by the synchronising calls
    // kernel timing hooks (qlga_profile_*)
    int prof_on;
    int prof_n;
    cudaEvent_t* prof_ev;  // [PROF_CAP], created on first enable
    signed char* prof_kind;
    char err[512];
};
constexpr int PROF_CAP = 4097;
