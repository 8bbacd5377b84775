/*
 * qlga.h -- C ABI of the B200-native spin-2 BEC quantum lattice gas (QLGA) step.
 *
 * Method: arXiv:1907.12834.  Five coupled Gross-Pitaevskii fields
 * psi_m (m_f = +2..-2, eq. 34/37), each carried by a pair of
 * spinor amplitudes per lattice site:  psi_m = q_m1 + q_m2.
 * One time step is the operator product of eq. (108) (plain) or eq. (112)
 * (interleaved), built from the kinetic factors
 * I'_i = S_i C S_i^T C of eq. (107) and the local interaction unitary U.
 * Where the paper is silent the readings R1..R11 of DESIGN.md apply.
 *
 * All entry points are plain C, take plain pointers and sizes, return a status
 * and never throw or abort.  Pointers are marked HOST or DEVICE below.  Device
 * buffers and the CUDA stream are owned by the caller (e.g. torch tensors and a
 * torch stream); the library only allocates small reduction / staging scratch
 * of its own and frees it in qlga_destroy.  All work is enqueued on the caller's
 * stream; calls that return data to the host synchronise that stream.
 *
 * Data layout (both for the caller's transfers and inside the device buffers):
 *   q   : [5][2][Nz][Ny][Nx] complex   index (((j*2 + sigma)*Nz + z)*Ny + y)*Nx + x
 *   psi : [5][Nz][Ny][Nx]    complex
 *   omega : [5][Ny][Nx]      real (2D only)
 *   j = 0..4 <-> m_f = +2,+1,0,-1,-2;  sigma = 0,1 <-> spinor component 1,2;
 *   x fastest; Ny = Nz = 1 in 1D, Nz = 1 in 2D; complex = interleaved (re, im) of the
 *   context's storage type (double for QLGA_F64, float for QLGA_F32 and QLGA_F32X); periodic in x, y, z.
 */
#ifndef QLGA_H
#define QLGA_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct qlga_ctx qlga_ctx;   /* opaque, owned by the library */

typedef enum {
    QLGA_OK = 0,
    QLGA_EINVAL = 1,   /* bad argument; no side effect                        */
    QLGA_ENOMEM = 2,   /* host or device allocation of library scratch failed */
    QLGA_ECUDA = 3,    /* CUDA error; text in qlga_last_error                 */
    QLGA_ESTATE = 4,   /* call not valid in the current state (no state set)  */
    QLGA_EUNSUP = 5    /* not supported for this context (e.g. vorticity in 1D) */
} qlga_status;

/* Precision of a context.
 *   QLGA_F64   state and arithmetic in fp64 (160 B per site); follows the oracle to rounding.
 *   QLGA_F32   state and arithmetic in fp32 (80 B per site): the throughput / memory variant.
 *   QLGA_F32X  state stored in fp32 (80 B per site, the same buffers and transfers as QLGA_F32), arithmetic in
 *              fp64 registers inside every pass: one rounding to fp32 per amplitude per pass instead of one per
 *              floating-point operation (measured error growth in DESIGN.md section 8). */
typedef enum { QLGA_F64 = 0, QLGA_F32 = 1, QLGA_F32X = 2 } qlga_prec;

/* Operator ordering of one time step (rightmost operator acts first):
 *   QLGA_PLAIN        eq. (108):  I'_x1 I'_x1 I'_x2 I'_x2 [I'_y1 I'_y1 I'_y2 I'_y2] U
 *   QLGA_INTERLEAVED  eq. (112):  every I' preceded by U^{1/(4 ndim)}, "n = 8" in 2D and
 *                                 "n = 12" in 3D.  Factors of z act first, then
 *                                 y, then x (R7). */
typedef enum { QLGA_PLAIN = 0, QLGA_INTERLEAVED = 1 } qlga_order;

/* Tunables of qlga_set_option. */
typedef enum {
    QLGA_OPT_PATH = 0,        /* 0 = fused pass kernels (default), 1 = one kernel per operator   */
    QLGA_OPT_STEPS_PER_LAUNCH = 1, /* 1D only: time steps fused per launch (halo 4 per step); 0 = auto, else 1..15,
                                 clamped to what the x pass's CTA size supports ((threads - 8) / 16) */
    QLGA_OPT_EXP_TOL_LOG2 = 2,/* truncation target of the interaction exponential, log2 (default -58 for QLGA_F64,
                                 -44 for QLGA_F32X, -27 for QLGA_F32) */
    QLGA_OPT_THREADS_X = 3,   /* CTA size of the x pass: 64, 96, 128, 192 or 256; 0 = auto       */
    QLGA_OPT_TILE_Y = 4,      /* strided (y, z) passes: columns per CTA (1,2,4,8); 0 = auto      */
    QLGA_OPT_THREADS_Y = 5,   /* CTA size of the strided passes; 0 = auto.  TILE_Y and THREADS_Y are validated as a
                                 pair: columns x threads 1x64, 1x96, 1x128, 1x192, 2x128, 2x192, 2x256, 4x256, 8x256
                                 (either one 0 = auto for that one); any other pair is QLGA_EINVAL when it is set, and a
                                 pair that only resolves to an unbuilt kernel at launch is QLGA_EINVAL from qlga_step */
    QLGA_OPT_FUSE_PLAIN_U = 6,/* plain ordering in 2D/3D, several steps per qlga_step call: 1 (default) = the U of
                                 step t+1 is applied at the end of step t's x pass (same operator product, no halo
                                 recompute of U, and it fills the memory-bound pass); 0 = always on the first pass */
    QLGA_OPT_F32_PHASE = 7,   /* QLGA_F32 only: formulation of the scalar phase factor exp(-i s (c0 rho + mu)):
                                 0 = (cos, -sin) rounded to fp32 (default), 1 = 1 + d with cos - 1 kept to its own
                                 precision, 2 = 1 + d with d evaluated in fp64 (measured: DESIGN.md section 8) */
    QLGA_OPT_EXP_POLY = 8,    /* interaction polynomial: 0 = Chebyshev-economised Taylor, 1 = plain Taylor */
    QLGA_OPT_MARCH = 10,      /* strided passes that carry no interaction (plain ordering): 1 (default) = column
                                 marching, one thread per (column, m_f), the four factors as a register pipeline, no
                                 shared memory (bit-identical results); 0 = the tile kernel.  Setting TILE_Y or
                                 THREADS_Y also selects the tile kernel */
    QLGA_OPT_BAND = 11,       /* plain ordering in 2D: ONE HBM round trip per time step by band pipelining.  The lattice is
                                 cut into bands of rows; the interaction-free y pass (marching kernel) of band k writes
                                 into a small ring buffer owned by the library that stays resident in the 126 MB L2, the
                                 x pass (with the next step's U) of band k reads it from there and writes the new state;
                                 the y pass of band k+1 runs beside the x pass of band k (the library's own streams,
                                 ordered by events).  Same kernels, same arithmetic: results are bit-identical to the
                                 two-launch step.  0 = off (a y-pass launch and an x-pass launch per step: two round
                                 trips), 1 = bands issued directly on the library's streams (host-bound; debugging), 2 =
                                 the band schedule of a step instantiated once as a CUDA graph and replayed with one
                                 cudaGraphLaunch on the caller's stream, -1 (default) = 2 where it pays: a band's x kernel
                                 still fills the GPU (rows per band x tiles per row >= 888) and the state is larger than
                                 256 MB.  Band mode applies to: 2D, QLGA_PLAIN, fused path, marching pass on, at least four
                                 bands, and every step of a qlga_step call whose U was applied by the step before it, i.e.
                                 all but the first and, with a third buffer, the last -- step in calls of many steps.
                                 Side effects of band mode: the library allocates the ring (slots x rows x Nx x 10 planes,
                                 63 MB at the defaults), creates four streams of its own, and raises the device's
                                 persisting-L2 set-aside (cudaLimitPersistingL2CacheSize, a per-device limit that stays
                                 raised) to the ring's size: the ring's lines are marked persisting so that the y pass's
                                 output is never written back to DRAM.  The first band step of a context allocates and
                                 captures (not to be called while the caller's stream is itself being captured) */
    QLGA_OPT_BAND_ROWS = 12,  /* rows per band; 0 = auto (about 20 MB per band) */
    QLGA_OPT_BAND_SLOTS = 13, /* bands the ring holds: 2..8; 0 = auto (3) */
    QLGA_OPT_EXP_MOD_SHIFT = 9 /* the MODULUS part of the truncation error (the even part of the polynomial) is held to
                                 2^(tol_log2 - shift): a modulus error that repeats at every application changes the
                                 density and with it the phase rate c0 rho, and grows like applications x (c0 rho t / 2)
                                 (DESIGN.md section 8).  0..16; default 7 for QLGA_F64 (modulus part 2^-65), 8 for QLGA_F32X (2^-52),
                                 0 for QLGA_F32 */
} qlga_option;

/* Lattice sums returned by qlga_observables (always double).
 *   n_m[j]   = sum_r |psi_m|^2                                   eq. (3)
 *   norm_psi = sum_m n_m ;  norm_q = sum_{r,m,sigma} |q|^2  (the unitary invariant)
 *   F[3]     = sum_r <psi|f_nu|psi>, nu = x,y,z                  eq. (5), (59)-(60)
 *   A00      = sum_r A00(r), A00(r) = (2 psi_2 psi_-2 - 2 psi_1 psi_-1 + psi_0^2)/sqrt(5)   eq. (4), (35)
 *   A00_abs2 = sum_r |A00(r)|^2
 *   e_kin    = sum_r sum_m sum_d |psi_m(r+e_d) - psi_m(r)|^2     (eq. 12 with hbar = 1, m = 1/2)
 *   e_c0, e_c1, e_c2 = (c0/2) sum rho^2, (c1/2) sum |F|^2, (c2/2) sum |A00|^2   eq. (32)
 *   e_total  = e_kin + e_c0 + e_c1 + e_c2
 *   e_dt     = i(<psi(t)|psi(t)> - <psi(t)|psi(t-tau)>)/<psi(t)|psi(t)>        eq. (85), PAPER.md:666;
 *              NaN unless the previous step's state is still held (see qlga_init).
 *   step     = number of time steps taken since the last qlga_set_state_*.        */
typedef struct {
    double n_m[5];
    double norm_psi, norm_q;
    double F[3];
    double A00_re, A00_im, A00_abs2;
    double e_kin, e_c0, e_c1, e_c2, e_total;
    double e_dt_re, e_dt_im;
    int64_t step;
} qlga_obs;

/* Create a context (BASELINE.json north_star "qlga_init").
 *   out        HOST  receives the context.
 *   ndim       1, 2 or 3.     dims  HOST  {Nx, Ny} (Ny must be 1 when ndim == 1) or, when
 *              ndim == 3, {Nx, Ny, Nz}; all >= 1.
 *   c0,c1,c2   the paper's g0, g1, g2 of eq. (32)-(34).
 *   dev_buf_a, dev_buf_b   DEVICE, caller-owned, 16-byte aligned, each >= qlga_state_bytes().
 *   dev_buf_c  DEVICE or NULL.  Optional third buffer: in 2D (3D) a step is two (three)
 *              passes, so the state of the previous step survives only with a third
 *              buffer; without it e_dt is NaN in 2D and 3D.  Unused in 1D.
 *   buf_bytes  size of each buffer.
 *   cuda_stream  the caller's cudaStream_t (NULL = legacy default stream); a stream of the device that holds the buffers.
 * The context lives on the device its buffers are on (all three on the same one), whatever device is current in the
 * calling thread: every entry point that takes the context switches to that device and restores the caller's on return.
 * Errors: QLGA_EINVAL (arguments), QLGA_ECUDA (no sm_100 device / CUDA failure), QLGA_ENOMEM. */
qlga_status qlga_init(qlga_ctx** out, int ndim, const int64_t* dims,
                      double c0, double c1, double c2, qlga_order order, qlga_prec prec,
                      void* dev_buf_a, void* dev_buf_b, void* dev_buf_c, size_t buf_bytes,
                      void* cuda_stream);

/* Bytes one state buffer needs: 10 * Nx * Ny * Nz * 2 * sizeof(real).  0 on bad arguments. */
size_t qlga_state_bytes(int ndim, const int64_t* dims, qlga_prec prec);

/* Set a tunable (see qlga_option).  QLGA_EINVAL for unknown keys / bad values. */
qlga_status qlga_set_option(qlga_ctx*, qlga_option key, int64_t value);

/* Load the bosonic field: q_m1 = q_m2 = psi_m / 2 (reading R6).  psi: HOST or DEVICE
 * ([5][Nz][Ny][Nx] complex of the context's storage type (double for QLGA_F64, float for QLGA_F32 and QLGA_F32X)) per src_on_device.  Resets step to 0. */
qlga_status qlga_set_state_psi(qlga_ctx*, const void* psi, int src_on_device);
/* Load / read back the full spinor state q ([5][2][Nz][Ny][Nx] complex); also the checkpoint format. */
qlga_status qlga_set_state_q(qlga_ctx*, const void* q, int src_on_device);
qlga_status qlga_get_state_q(qlga_ctx*, void* q, int dst_on_device);
/* Read back psi_m = q_m1 + q_m2. */
qlga_status qlga_get_state_psi(qlga_ctx*, void* psi, int dst_on_device);

/* Chemical potential term mu psi_m of the equation of motion (section II.C;
 * dispersion relations eq. 75): H_int + mu 1, one more scalar phase
 * exp(-i s mu) in every U^(s).  Default 0 (the paper's own simulations).  Takes effect from the next
 * qlga_step.  QLGA_EINVAL for a non-finite value. */
qlga_status qlga_set_chemical_potential(qlga_ctx*, double mu);

/* Advance n >= 0 time steps of eq. (108)/(112).  Asynchronous on the stream. */
qlga_status qlga_step(qlga_ctx*, int64_t n);

/* Lattice sums of the current state; host_out HOST.  Synchronises the stream. */
qlga_status qlga_observables(qlga_ctx*, qlga_obs* host_out);

/* Lattice vorticity, 2D only (eq. 99-104, reading R8), per m:
 *   v_x(r) = (1/2) arg(psi(r+e_x) psi*(r-e_x)),  v_y(r) = (1/2) arg(psi(r+e_y) psi*(r-e_y)),
 *   omega(r) = (1/2)[v_y(r+e_x) - v_y(r-e_x) - v_x(r+e_y) + v_x(r-e_y)],   arg(0) := 0.
 * omega: HOST or DEVICE [5][Ny][Nx] real of the context's storage type.  QLGA_EUNSUP in 1D. */
qlga_status qlga_vorticity(qlga_ctx*, void* omega, int dst_on_device);

/* Interaction-angle statistics of the current state (diagnostic; it tells which polynomial degrees and
 * which code path of U a state exercises).  For one application of U^(s) (s = 1 plain, 1/(4 ndim)
 * interleaved, eq. 108 / 112) at every site:
 *   theta = s (2 |c1| |F| + (|c2|/5) rho)   the spectral-norm bound of s K the kernels select the degree by,
 *   phase = |s (c0 rho + mu)|               the scalar phase.
 * host_out HOST: theta_max, theta_mean (atomic accumulation: reproducible to rounding only), phase_max,
 * degree_hist[p] = number of sites whose own angle takes polynomial degree p = 1..12 by the kernels' lookup
 * ([0] = sites beyond the split angle, which take the general path).  Synchronises the stream. */
typedef struct { double theta_max, theta_mean, phase_max; int64_t degree_hist[13]; } qlga_angles;
qlga_status qlga_angle_stats(qlga_ctx*, qlga_angles* host_out);

/* Total density rho(r) = sum_m |psi_m(r)|^2 = psi psi^dagger; rho: HOST or DEVICE [Nz][Ny][Nx] real. */
qlga_status qlga_density(qlga_ctx*, void* rho, int dst_on_device);

/* L2 error of eq. (115), PAPER.md:1074 (the paper's convergence measure, Figs. 23-24):
 *   *host_eps = sum_r (rho_ref(r) - rho(r))^2,  rho_ref: HOST or DEVICE [Nz][Ny][Nx] real of the
 * context's storage type (e.g. the density of the initial eigenstate).  Synchronises the stream. */
qlga_status qlga_density_l2_error(qlga_ctx*, const void* rho_ref, int src_on_device, double* host_eps);

/* Vortex detection, 2D only (the paper tracks vortices of positive / negative winding number,
 * Figs. 18, 21, 22; detector = reading R15 of DESIGN.md): winding number of
 * every elementary plaquette, corners counter-clockwise a=(x,y), b=(x+1,y), c=(x+1,y+1), d=(x,y+1),
 *   w = [arg(b a*) + arg(c b*) + arg(d c*) + arg(a d*)] / (2 pi)  in {-1, 0, +1}   (arg(0) := 0),
 * per m.  Writes up to max_out records (j, x, y, w) of the plaquettes with w != 0 to
 * host_out (HOST, int32 [max_out][4], order unspecified) and the total number found to
 * *host_count (may exceed max_out).  Synchronises the stream.  QLGA_EUNSUP in 1D. */
qlga_status qlga_vortices(qlga_ctx*, int32_t* host_out, int64_t max_out, int64_t* host_count);

/* Vortex tracking, 2D only: association of two detections (the paper follows vortices of positive / negative
 * winding as tracks, Figs. 18, 21, 22; the tracker is not printed: reading R18 of DESIGN.md).
 * host_prev / host_cur: HOST int32 [n][4] records (j, x, y, w) as written by qlga_vortices at two times.  Two
 * records can be the same vortex only if they agree in j and w.  With d2 the periodic (minimal-image) squared
 * lattice distance, the nearest candidate of a record is the record of the other list with the same (j, w)
 * and d2 <= max_dist2 that minimises (d2, y, x) lexicographically; two records are matched iff each is the
 * other's nearest candidate.  host_match_cur[i] = index into prev of the match of cur[i], or -1 (a vortex that
 * appeared); host_match_prev[k] = index into cur, or -1 (a vortex that disappeared: annihilation with a partner of
 * opposite winding, or a jump beyond max_dist2).  At most QLGA_MATCH_MAX records per list.  The O(n_prev n_cur)
 * search runs on the device.  Synchronises the stream.  QLGA_EINVAL (arguments, a record outside the lattice),
 * QLGA_EUNSUP (not 2D). */
#define QLGA_MATCH_MAX 65536
qlga_status qlga_vortex_match(qlga_ctx*, const int32_t* host_prev, int64_t n_prev, const int32_t* host_cur,
                              int64_t n_cur, int64_t max_dist2, int32_t* host_match_cur, int32_t* host_match_prev);

/* ---- Slab decomposition over several GPUs ---------------------
 * The paper only states that its code "naturally scales with the number of GPUs"
 * (PAPER.md:1092-1094).  Here the lattice is cut into slabs along its slowest axis (x in 1D,
 * y in 2D, z in 3D), one slab per GPU / context.  A slab context is an ordinary context whose
 * slowest axis holds `ghost` ghost layers, then the owned layers, then `ghost` ghost layers.
 * A time step moves information by exactly 4 sites per direction (four kinetic factors of
 * radius 1), so with ghost = 4 valid ghost layers before a step the owned layers are exact
 * after it, whatever the periodic wrap of the extended slab puts into its ghost layers; the
 * ghost layers are then refreshed from the neighbouring slabs' edge layers (one exchange of
 * 2 x ghost x 160 B per site of a layer per step in fp64).  The library moves layers between
 * the state and contiguous DEVICE buffers; the transport between GPUs (NCCL send/recv, peer
 * copies) belongs to the caller.
 *
 * qlga_slab_configure: declare `ghost` (>= 0; 0 = not a slab) ghost layers on each side of the
 *   slowest axis; needs extent >= 3 * ghost.  The lattice sums (qlga_observable_sums,
 *   qlga_observables) then run over the owned layers only; the per-site maps (vorticity,
 *   density, vortices, state read-back) still cover the whole extended slab.
 * qlga_slab_edge_get: copy the `ghost` lowest (side 0) or highest (side 1) OWNED layers of all
 *   10 planes to dev_out, DEVICE [10][ghost][layer sites] complex.  Asynchronous on the stream.
 * qlga_slab_ghost_set: overwrite the low (side 0) or high (side 1) GHOST layers from dev_in
 *   (same layout).  Asynchronous on the stream.
 * Errors: QLGA_EINVAL (bad side / ghost, NULL), QLGA_ESTATE (no state, or not a slab). */
qlga_status qlga_slab_configure(qlga_ctx*, int64_t ghost);
qlga_status qlga_slab_edge_get(qlga_ctx*, int side, void* dev_out);
qlga_status qlga_slab_ghost_set(qlga_ctx*, int side, const void* dev_in);

/* The additive lattice sums behind qlga_observables, so that slabs can be added up before the
 * derived quantities are formed: host_sums HOST [QLGA_NSUMS] =
 *   n_m[5], sum|q|^2, F_x, F_y, F_z, Re A00, Im A00, sum|A00|^2, e_kin, sum rho^2, sum|F|^2,
 *   Re<psi(t)|psi(t-tau)>, Im<psi(t)|psi(t-tau)>  (the last two are NaN without a previous state).
 * Synchronises the stream.  qlga_observables_from_sums forms the qlga_obs record from such
 * sums (of one context or added over slabs); it launches nothing. */
#define QLGA_NSUMS 17
qlga_status qlga_observable_sums(qlga_ctx*, double* host_sums);
qlga_status qlga_observables_from_sums(const qlga_ctx*, const double* host_sums, qlga_obs* host_out);

/* Kernel timing hooks (used by bench.py for the roofline of the dominant kernel).
 * While enabled, qlga_step records a CUDA event on the caller's stream before every
 * pass kernel and one after the last; qlga_profile_read synchronises the stream,
 * returns the summed durations and launch counts per kernel kind since the last
 * read (0: x pass, 1: y pass, 2: per-operator kernels, 3: whole time steps in band mode,
 * QLGA_OPT_BAND, where the two passes run beside each other) and resets them.  At most
 * 4096 launches are recorded between two reads; later ones are not timed. */
typedef struct { double ms[4]; int64_t launches[4]; } qlga_profile;
qlga_status qlga_profile_enable(qlga_ctx*, int on);
qlga_status qlga_profile_read(qlga_ctx*, qlga_profile* host_out);

/* The polynomial the kernels use for the interaction exponential (host only, needs no GPU):
 * exp(-i s K) v = P_p(y) v, y = -i s K, P_p(y) = b0 (1 + r[1] y (1 + r[2] y (... (1 + r[p] y)))),
 * the Chebyshev-economised Taylor polynomial of degree p, valid for ||s K|| <= *theta_max within
 * 2^tol_log2, its even (modulus) part within 2^(tol_log2 - mod_shift) (mod_shift as
 * QLGA_OPT_EXP_MOD_SHIFT).  p = 1..12.  Exposed so that the table can be tested on the CPU. */
qlga_status qlga_exp_polynomial(int tol_log2, int mod_shift, int p, double* theta_max, double* b0, double* r);
/* The degree the kernels pick for a (warp-uniform) angle theta <= min(theta_max of degree 12, 1/2): a table
 * lookup on the exponent and the top four mantissa bits of theta as a float, whose entry serves the upper
 * edge of its bucket -- never below "smallest p with theta <= theta_max(p)", at most one above (host only). */
qlga_status qlga_exp_degree(int tol_log2, int mod_shift, double theta, int* p);

/* The lattice sums of qlga_observable_sums for callers that cannot allocate device memory (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Needs NO context (qlga_init allocates
 * its scratch with cudaMalloc) and calls no cudaMalloc / cudaFree or allocating routine: the per-block partial
 * sums live in a static device array inside the library, 19 doubles for each of at most
 * QLGA_NOALLOC_MAX_BLOCKS = 2048 blocks plus 19 reduced sums = 311 448 bytes, held by every GPU that loads the
 * library until the process exits.
 *   dev_q      DEVICE  state [5][2][Nz][Ny][Nx] complex of the storage type of `prec` (layout at the top)
 *   dev_qprev  DEVICE or NULL  the previous step's state, for the two sums of eq. (85)
 *   ndim, dims as for qlga_init;  prec: QLGA_F64, or QLGA_F32 / QLGA_F32X (fp32 storage)
 *   nblocks    grid of the reduction: 0 = the grid qlga_observable_sums uses (8 per SM), else 1..2048;
 *              a value beyond QLGA_NOALLOC_MAX_BLOCKS is QLGA_EINVAL (the static scratch cannot hold it)
 *   dev_sums   DEVICE [QLGA_NSUMS] doubles, the caller's: the sums in the order of qlga_observable_sums (whole
 *              lattice); entries 15, 16 are 0 when dev_qprev is NULL
 *   cuda_stream  the caller's stream; asynchronous, no synchronisation, no host output
 * With the same grid the sums equal qlga_observable_sums' bit for bit (same kernels).  All calls share the one
 * array (nothing in it needs clearing between calls): calls that may overlap on the GPU -- different streams
 * without an ordering between them -- race; keep them on one stream or order them with events.
 * Errors: QLGA_EINVAL (arguments, nblocks > 2048), QLGA_EUNSUP (device ordinal > 63), QLGA_ECUDA; the text is
 * returned by qlga_noalloc_last_error(). */
#define QLGA_NOALLOC_MAX_BLOCKS 2048
qlga_status qlga_observable_sums_noalloc(const void* dev_q, const void* dev_qprev, int ndim, const int64_t* dims,
                                         qlga_prec prec, int nblocks, double* dev_sums, void* cuda_stream);
const char* qlga_noalloc_last_error(void);

/* Issue rate of the plain floating-point pipes, measured (the denominator of bench.py's "alu" roofline;
 * SURVEY.md 8(d)): a kernel of independent chains of one instruction kind, kind = 0 DFMA (fp64), 1 FFMA (fp32),
 * 2 FFMA2 (packed two-wide fp32), at 1024 resident threads per SM on the current device and the given stream
 * (cuda_stream = the caller's cudaStream_t or NULL).  *instr_per_s: thread-instructions per second (one per
 * lane; an FFMA2 counts as two) by CUDA events, best of three launches; *instr_per_clk_per_sm: the same per SM
 * cycle by clock64() (independent of the clock the GPU held); *ms (may be NULL): duration of the best launch.
 * Needs no context.  Synchronises the stream.  QLGA_EINVAL (kind, NULL), QLGA_ECUDA. */
qlga_status qlga_issue_peak(int kind, void* cuda_stream, double* instr_per_s, double* instr_per_clk_per_sm, double* ms);

/* Number of kernels this context has launched so far (for bench.py's gpu_launches). */
int64_t qlga_launch_count(const qlga_ctx*);

/* Text of the last error of this context (or of the failed qlga_init when ctx == NULL).
 * Owned by the library; valid until the next call on the same context. */
const char* qlga_last_error(const qlga_ctx*);

/* Free the context and the library's scratch.  Never frees caller buffers. */
qlga_status qlga_destroy(qlga_ctx*);

/* Library version string, e.g. "qlga-b200 0.1 (sm_100a)". */
const char* qlga_version(void);

#ifdef __cplusplus
}
#endif
#endif /* QLGA_H */
