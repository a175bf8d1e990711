/*
 * tcp.h -- C ABI of the B200-native thermocapillary central-moment phase-field lattice Boltzmann
 * step (arxiv 2401.03041; citations are PAPER.md:<line> of the reference text).
 *
 * One `tcp_sim` holds the state of one simulation on one GPU: the post-collision populations
 * h~ (D3Q27, phase field, eq. 10), g~ (D3Q27, hydrodynamics, eq. 16),
 * f~ (D3Q7/15/19/27, temperature, eq. 27; absent on the Runge-Kutta paths) and the
 * fields phi, u, T.  `tcp_step` advances it by Algorithm 1 / Algorithm 2.
 *
 * Conventions
 *   - cell index = x + nx*(y + ny*z), x fastest; every cell is fluid; a WALLS axis has no-slip,
 *     fixed-temperature walls half a cell outside its first and last cell.
 *   - arrays are in the simulation's precision (double for TCP_F64, float for TCP_F32);
 *     vector fields are 3 planes [3][nz][ny][nx].
 *   - array arguments may be HOST or DEVICE pointers (resolved with cudaMemcpyDefault); the
 *     caller owns them, the library copies.  Wall planes: axis 0 -> [nz][ny], 1 -> [nz][nx],
 *     2 -> [ny][nx].
 *   - every function returns TCP_OK (0) or a negative TCP_E* code, never throws or aborts;
 *     `tcp_last_error()` gives a thread-local message for the last failure on this thread.
 *   - there is no CPU fallback: without a CUDA device every call that needs one fails with
 *     TCP_ECUDA.
 */
#ifndef TCP_H
#define TCP_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tcp_sim tcp_sim; /* opaque; owned by the library; freed by tcp_destroy */

enum { TCP_OK = 0, TCP_EINVAL = -1, TCP_ENOMEM = -2, TCP_ECUDA = -3, TCP_EUNSUPPORTED = -4, TCP_ESTATE = -5 };
enum { TCP_F64 = 0, TCP_F32 = 1 };
enum { TCP_THERMAL_LB_D3Q7 = 0, TCP_THERMAL_LB_D3Q15, TCP_THERMAL_LB_D3Q19, TCP_THERMAL_LB_D3Q27,
       TCP_THERMAL_RK2, TCP_THERMAL_RK4 };
enum { TCP_BC_PERIODIC = 0, TCP_BC_WALLS = 1 };
enum { TCP_STREAM_TWO_GRID = 0, TCP_STREAM_AA = 1 };
enum { TCP_SPACE_CENTRAL = 0, TCP_SPACE_RAW = 1 };
enum { TCP_EQ_SECOND_ORDER = 0, TCP_EQ_MAXWELLIAN = 1 };   /* equilibria: eqs. 12 / 18 as printed, or the Maxwellian in central-moment space */   /* collision space: central moments (the paper's model) or raw moments (MRT) */ /* AA: in place, one grid of populations (half the memory) */

/* The paper's problem statement (sections 2.1-2.3).  Fill `struct_size = sizeof(tcp_params)`. */
typedef struct tcp_params {
    unsigned struct_size;
    int precision;                     /* TCP_F64 | TCP_F32 */
    int thermal;                       /* TCP_THERMAL_*: eqs. 27-29 (LB) or eqs. 25-26 with eq. 4 (RK) */
    int streaming;                     /* TCP_STREAM_* */
    int bc[3];                         /* TCP_BC_* for x, y, z */
    double rho_H, rho_L;               /* eq. 14 */
    double tau_H, tau_L;               /* eq. 22; nu = tau c_s^2, rate 1/(tau+1/2) */
    double xi, M;                      /* interface width, mobility: eqs. 3, 11, 15 */
    double sigma_ref, sigma_T, T_ref;  /* eq. 9 */
    double kappa_H, kappa_L, cp_H, cp_L; /* eqs. 23-24; rho and c_p enter only the RK paths (eq. 4) */
    double gravity[3];                 /* eq. 7 */
    double wall_T[3][2];               /* constant wall temperature per axis / face (eqs. 30-31) */
    double s_bulk, s_high;             /* central-moment rates of the trace of the 2nd-order moments and of
                                          all moments of order >= 3 (hydrodynamic lattice); default 1, 1.
                                          s_high = 1 runs the closed-form collision, any other value the
                                          full central-moment transform (about 25 % more instructions) */
    int high_rate_equals_shear;        /* 1: every rate = the physical one = plain BGK + Guo */
    double eps_normal;                 /* n = grad phi / sqrt(|grad phi|^2 + eps); default 1e-32 */
    double wall_u[3][2][3];            /* velocity of each wall [axis][face][component] (moving wall):
                                          enters the bounce-back of g only; default 0 */
    double sigma_TT;                   /* d^2 sigma / dT^2 of a parabolic sigma(T) = sigma_ref + sigma_T (T - T_ref)
                                          + sigma_TT (T - T_ref)^2 / 2 (self-rewetting fluids); the
                                          Marangoni term of eq. 8 then carries d sigma/dT = sigma_T + sigma_TT (T - T_ref).
                                          Default 0 = eq. 9 as printed */
    double wall_contact_angle[3][2];   /* wetting boundary condition (refs. [34], [35]): contact angle of each wall
                                          [axis][face] in degrees, 0..180, measured inside the phi = 1 fluid.  The ghost value of
                                          phi behind the wall follows from n_w . grad phi = -(4 / xi) cos(theta) phi_w (1 - phi_w)
                                          with phi_w = (phi_f + phi_g) / 2 at the wall half a cell outside the first cell:
                                          a phi_w^2 - (1 + a) phi_w + phi_f = 0, a = -(2 / xi) cos(theta), phi_g = 2 phi_w - phi_f.
                                          Default 90 = neutral wetting = mirror ghost */
    int hydro_lattice;                 /* lattice of the hydrodynamic populations g: 27 (default) or 19 ("hydrodynamic LBM solvers
                                          often rely on a D3Q19 or D3Q27 stencil"; weights eq. B.3, central-moment
                                          basis x^a y^b z^c with a, b, c <= 2 and abc = 0).  19 moves 16 values per cell less
                                          (928 instead of 1056 B with the D3Q7 thermal LB); collisions: s_high = 1 or BGK only */
    int collision_space;               /* TCP_SPACE_CENTRAL (default): moments about the local velocity; TCP_SPACE_RAW: the same
                                          basis and rates about the lattice at rest, i.e. the multiple-relaxation-time (MRT) operator
                                          ("the SRT or MRT methods retain widespread usage").  With
                                          high_rate_equals_shear = 1 (SRT / BGK) the two coincide.  Same kernels, same cost */
    int equilibrium;                   /* TCP_EQ_SECOND_ORDER (default): eqs. 12 and 18 as printed; TCP_EQ_MAXWELLIAN: the continuous
                                          Maxwell-Boltzmann distribution taken in central-moment space (central moments of x^a y^b z^c
                                          = s m_a m_b m_c, m = (1, 0, c_s^2); on D3Q27 the product form), in place of eq. 12; eq. 18
                                          becomes w_i (p* - 1) + that equilibrium with s = 1.  Moments up to second order are
                                          unchanged.  D3Q27 lattices only: hydro_lattice = 27 and thermal D3Q27 LB / RK2 / RK4; closed-form
                                          collision only (s_high = 1, high_rate_equals_shear = 0); either collision space */
} tcp_params;

/* Fill *p with the defaults: struct_size, fp64, thermal LB D3Q7, two-grid, periodic x 3, rho = 1, tau = 0.6, xi = 4,
 * M = 0.05, sigma = 0, kappa = 0.2, c_p = 1, no gravity, walls at rest, at T = 0 and neutrally wetting (90 degrees), s_bulk = s_high = 1 (the closed-form
 * central-moment collision), eps_normal = 1e-32, hydro_lattice = 27.  A zero-initialised struct is NOT valid (eps_normal = 0 makes the
 * interface normal 0/0 in the bulk, s_bulk = s_high = 0 are not relaxation rates): tcp_create rejects it with TCP_EINVAL.
 * Errors: TCP_EINVAL (p NULL). */
int tcp_params_default(tcp_params *p);

/* Bytes of device memory one simulation needs (populations, fields, wall planes).
 * Errors: TCP_EINVAL (bad extents / parameters), TCP_EUNSUPPORTED. */
int tcp_workspace_bytes(int nx, int ny, int nz, const tcp_params *p, size_t *bytes);

/* Create a simulation; the library allocates the workspace (cudaMalloc) and a stream.
 * Validation: n >= 1 (>= 2 on WALLS axes), nx*ny*nz <= 429 496 729 (32-bit offsets within a group of 9 population planes), tau > -1/2, M, xi, rho, kappa, cp, eps_normal > 0, 0 < s_bulk, s_high < 2.
 * The simulation lives on the CUDA device that is current at the call; every later call makes that device current
 * for its own duration, so simulations on several GPUs can be driven from one thread.
 * Errors: TCP_EINVAL, TCP_EUNSUPPORTED, TCP_ENOMEM, TCP_ECUDA. */
int tcp_create(int nx, int ny, int nz, const tcp_params *p, tcp_sim **out);

/* Same, on caller-owned device memory (>= tcp_workspace_bytes, 256-byte aligned) and on the
 * caller's CUDA stream (a cudaStream_t passed as void*; NULL = default stream).  The memory and
 * the stream must outlive the simulation.  The simulation lives on the device that owns the workspace (resolved with
 * cudaPointerGetAttributes); the stream must belong to the same device. */
int tcp_create_in(int nx, int ny, int nz, const tcp_params *p, void *dev_workspace, size_t bytes,
                  void *cuda_stream, tcp_sim **out);

/* Set phi, u, T and initialise all populations to their equilibria:
 * h~ = h_eq(phi, u) (eq. 12), g~ = g_eq(p* = 0, u) (eq. 18), f~ = f_eq(T, u).
 * u == NULL -> 0; T == NULL -> T_ref.  Errors: TCP_EINVAL (phi NULL), TCP_ECUDA. */
int tcp_init_fields(tcp_sim *s, const void *phi, const void *u, const void *T);

/* Per-wall-cell Dirichlet temperature (eq. 30); Tw == NULL restores the constant wall_T.  May be called at any time
 * between steps; the new plane acts from the next step on, identically for both streaming patterns (with TCP_STREAM_AA
 * the wall links that are stored already anti-bounced are corrected for the change). */
int tcp_set_wall_temperature(tcp_sim *s, int axis, int face, const void *Tw);

/* Volumetric heat source q_T [nz][ny][nx] of eqs. 4 / 27 (e.g. eq. 37); NULL (default) = none. */
int tcp_set_heat_source(tcp_sim *s, const void *q);

/* Advance nsteps time steps: per step, the phase-field update (eqs. 10-15), the hydrodynamic
 * update (eqs. 16-22 with the forces of eqs. 7-9) and the temperature update (eqs. 27-29, or
 * eq. 4 by eq. 26 / eq. 25).  Asynchronous on the simulation's stream.
 * Errors: TCP_ESTATE (fields not initialised), TCP_EINVAL (nsteps < 0), TCP_ECUDA. */
int tcp_step(tcp_sim *s, int nsteps);

/* Temperature pre-initialisation (the temperature field is often initialised by running the
 * thermal solver to convergence): nsteps temperature updates alone (thermal LB, or the RK stages), with phi,
 * u and the phase-field / hydrodynamic populations frozen.  With TCP_STREAM_AA and a thermal LB nsteps must
 * be even.  Errors: TCP_ESTATE, TCP_EINVAL, TCP_ECUDA. */
int tcp_relax_temperature(tcp_sim *s, int nsteps);

/* ---- block decomposition along z ("the domain is partitioned into blocks ... ghost layers";
 * Algorithm 1 updates the cells next to a block face first and sends their populations while the interior is
 * updated).  A slab is an ordinary simulation whose z-plane 0 (`lo`) and / or z-plane nz-1 (`hi`) is a GHOST
 * plane: it holds a copy of the neighbouring slab's boundary plane, is never updated by this simulation, and
 * takes the place of the periodic wrap / wall of bc[2] on that face (a face without ghost plane keeps bc[2]).
 * Arrays passed to tcp_init_fields / tcp_set_heat_source / returned by tcp_read_fields include the ghost
 * planes (initial phi, T there = the neighbour's values; p is undefined there); wall-temperature planes of the
 * x and y walls include the ghost rows.  Two-grid streaming only (TCP_EUNSUPPORTED with TCP_STREAM_AA).
 *
 * A step has `tcp_halo_phases` phases, each followed by one message per face: 1 on the thermal LB paths (the
 * fused kernel; message [9 h~ planes][9 g~ planes][1, 5, 5 or 9 f~ planes][phi][T], nx*ny values each), 3 / 5 on
 * the RK2 / RK4 paths (Algorithm 2: the fused phase + hydro kernel with message [9 h~][9 g~][phi], then every
 * Runge-Kutta stage with its output plane as message, because the next stage differentiates it).  With
 * kappa_H = kappa_L the first stage runs inside the fused kernel (grad kappa . grad T vanishes and everything else
 * it needs is already in the cell's thread): one phase less (2 / 4), and the first message also carries the
 * plane of the first stage's output ([9 h~][9 g~][phi][Y1]).
 * `tcp_halo_message_bytes` gives the size of a phase's message, `tcp_halo_bytes` that of the largest (phase 0).
 * `send_*` / `recv_*` are caller-owned DEVICE buffers of tcp_halo_bytes (NULL for a face without ghost plane);
 * `comm_stream` is the caller's cudaStream_t on which the library gathers and scatters and on which the caller
 * must enqueue, after every phase, the transfer of the first tcp_halo_message_bytes of send_hi -> the upper
 * neighbour's recv_lo and of send_lo -> the lower neighbour's recv_hi.  lo = hi = 0 makes it a plain box again. */
int tcp_set_halo(tcp_sim *s, int lo, int hi, void *comm_stream, void *send_lo, void *send_hi, void *recv_lo,
                 void *recv_hi);
int tcp_halo_phases(const tcp_sim *s, int *phases);
int tcp_halo_message_bytes(const tcp_sim *s, int phase, size_t *bytes);
int tcp_halo_bytes(const tcp_sim *s, size_t *bytes);

/* One time step of a slab: tcp_step_begin, then, after each transfer, tcp_step_advance until it reports 0
 * transfers left.  tcp_step_begin runs phase 0: its kernel on the plane(s) next to a ghost plane (simulation's
 * stream), then -- on comm_stream, as soon as those are done -- the gather of their new values into send_lo /
 * send_hi, and on the simulation's stream the same kernel on the interior planes.  tcp_step_advance scatters
 * recv_lo / recv_hi into the ghost planes (comm_stream, i.e. after the transfer the caller enqueued there; the
 * simulation's stream then waits for it) and either runs the next phase the same way (*transfers_left >= 1) or
 * completes the step (*transfers_left = 0).  tcp_step_end = the tcp_step_advance that completes the step
 * (TCP_ESTATE if phases remain; all a thermal LB slab needs).  All asynchronous.  tcp_step returns TCP_ESTATE
 * on a slab; these return TCP_ESTATE on a plain box or when called out of order. */
int tcp_step_begin(tcp_sim *s);
int tcp_step_advance(tcp_sim *s, int *transfers_left);
int tcp_step_end(tcp_sim *s);

/* Copy out phi, u, p = c_s^2 rho(phi) sum_i g~_i, T; any pointer may be NULL.
 * Synchronises the stream. */
int tcp_read_fields(tcp_sim *s, void *phi, void *u, void *p, void *T);

/* The pressure read-back of tcp_read_fields for callers that must not allocate (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): p = c_s^2 rho(phi) sum_i g~_i into `p` (HOST or
 * DEVICE pointer, nx*ny*nz values in the simulation's precision).  tcp_read_fields stages p in a spare buffer of the
 * workspace; this call stages it in a file-scope `static __device__` array of TCP_STATIC_SCRATCH_BYTES (8 MiB) that every
 * GPU which loads the library holds until the process exits, and calls no cudaMalloc, cudaFree or allocating library
 * routine.  Limit: nx*ny*nz * sizeof(real) <= TCP_STATIC_SCRATCH_BYTES, i.e. 2^20 cells in fp64 and 2^21 in fp32
 * (BASELINE configs 1 and 2, boxes up to 101^3 / 128^3); anything larger returns TCP_EUNSUPPORTED -- use tcp_read_fields.
 * The array is shared by every simulation and every call on that GPU and keeps the last call's contents; the kernel
 * overwrites all of its first nx*ny*nz entries before they are copied out, so nothing has to be cleared.  The call
 * returns after the copy has completed (it synchronises the simulation's stream), so calls made one after the other from
 * one thread are safe; calls that overlap on the GPU (several host threads, simulations on different streams) race on the
 * array and must be serialised by the caller.
 * Errors: TCP_EINVAL (NULL), TCP_ESTATE (not initialised, or between tcp_step_begin and tcp_step_end),
 * TCP_EUNSUPPORTED (box larger than the array), TCP_ECUDA. */
#define TCP_STATIC_SCRATCH_BYTES (8u << 20)
int tcp_read_pressure_static(tcp_sim *s, void *p);

/* Wait for all work of this simulation.  Errors: TCP_ECUDA (incl. asynchronous kernel faults). */
int tcp_synchronize(tcp_sim *s);

/* Number of kernels this simulation has launched so far (bench.py's gpu_launches). */
long long tcp_launch_count(const tcp_sim *s);

/* Time the last tcp_step call spent on the device, in milliseconds, measured with CUDA events
 * recorded on the simulation's stream around the kernels of that call (synchronises).
 * Errors: TCP_ESTATE if tcp_step has not been called. */
int tcp_last_step_ms(tcp_sim *s, float *ms);

/* Roofline calibration, not part of the method: launch `nlaunches` times a kernel with exactly the memory
 * access pattern and staging of the fused step (same pulls, same stores) but no stencils and no collision,
 * and return its mean duration.  It reads the current state and overwrites only the spare grid and the
 * spare phi / T buffers, so the simulation is unchanged -- except u, which is rewritten with itself.
 * It times itself with events of its own and is not counted by tcp_launch_count, so tcp_last_step_ms and
 * tcp_launch_count keep describing the method's kernels only.
 * Errors: TCP_ESTATE, TCP_EINVAL, TCP_EUNSUPPORTED (walls, AA streaming, ghost planes, hydro_lattice = 19). */
int tcp_pattern_copy_ms(tcp_sim *s, int nlaunches, float *ms);

int tcp_destroy(tcp_sim *s);

const char *tcp_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* TCP_H */
