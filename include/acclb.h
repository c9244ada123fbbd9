/*
 * acclb.h -- C ABI of libacclb.so: the per-time-step lattice update of accLB (arXiv 2505.01126) on one
 * NVIDIA B200 (sm_100a).  Citations are PAPER.md:Lnn (+ equation) of /root/reference/PAPER.md; "Rnn" are the
 * readings of the paper listed in DESIGN.md section 2.
 *
 * What the library computes (one step t -> t+1, fully periodic box, lattice units dx = dt = 1, fp64):
 *   thread-safe regularized D3Q27 lattice-Boltzmann collide+stream of the hydrodynamic populations
 *     f_i(x + c_i, t+1) = f_i^eq + (1 - omega) f_i^neq + S_i / 2                 PAPER.md:L85  (Eq. 6)
 *   with the pressure-based equilibrium and second-order Hermite reconstruction  PAPER.md:L88-92 (Eq. 7)
 *   and Guo forcing S_i                                                          PAPER.md:L79  (Eq. 5),
 *   coupled (two_phase = 1) to the conservative Allen-Cahn equation              PAPER.md:L61  (Eq. 3)
 *   discretised with WENO5 advection and lattice stencils
 *   and to the interface force F = F^s + F^p + F^nu                              PAPER.md:L100 (Eq. 8).
 *
 * Conventions
 *   - Plain pointers and sizes only.  Every pointer argument says HOST or DEVICE.
 *   - Field layout: scalars [nz][ny][nx] with x fastest; vectors [3][nz][ny][nx], component 0 = x.
 *   - "rho" in this API is the zeroth moment p* = sum_i f_i (the conserved "mass", R19); the mixture density
 *     is rho(phi) = rho_g + (rho_l - rho_g) phi.
 *   - The library never allocates or frees device memory: the caller (PyTorch) passes ONE workspace block of
 *     accLB_workspace_bytes() bytes, 256-byte aligned, that must outlive the context.  It never frees caller
 *     memory.  All work is enqueued on params.stream of device params.device.
 *   - Return value 0 = ACCLB_OK, negative = error; accLB_last_error() gives the text (thread-local).
 *   - A context is not thread-safe; distinct contexts are independent (replicas across GPUs; or z-slabs of one domain
 *     whose halo planes the caller exchanges between steps, see accLB_halo_chunks).
 *   - There is no CPU fallback: every entry point needs a CUDA device.
 */
#ifndef ACCLB_H
#define ACCLB_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ACCLB_OK 0
#define ACCLB_EINVAL (-1)     /* bad size / parameter / NULL pointer                      */
#define ACCLB_EWORKSPACE (-2) /* workspace too small or not 256-byte aligned              */
#define ACCLB_ECUDA (-3)      /* CUDA runtime / launch error, text in accLB_last_error()  */
#define ACCLB_ENUMERIC (-4)   /* a diagnostic is not finite                               */

#define ACCLB_NDIAG 9 /* length of the accLB_diagnostics vector */

typedef struct accLB_ctx accLB_ctx; /* opaque; owned by the library; freed by accLB_destroy */

/* POD, copied at create; no pointer is kept except `stream`. */
typedef struct {
  double tau;       /* relaxation time > 0.5; nu = (tau - 1/2)/3, omega = 1/tau      */
  int two_phase;    /* 0: single component (rho == 1, phi ignored); 1: LB + Allen-Cahn   */
  double rho_l;     /* density where phi = 1 (R16)     */
  double rho_g;     /* density where phi = 0                                                               */
  double sigma;     /* surface tension gamma */
  double mobility;  /* D of Eq. 3 (BASELINE "M")      */
  double width;     /* interface width delta (BASELINE "W"); kappa = 4 D / delta      */
  int force_type;   /* 0 none | 1 ABC: A(sin kz + cos ky, sin kx + cos kz, sin ky + cos kx) PAPER.md:L167
                       | 2 sine: F0 (sin ky, sin kz, sin kx) (BASELINE config 2); R20                      */
  double force_amp; /* A or F0 (a force density: divided by rho(phi) like the other forces, R3)            */
  int force_k;      /* forcing wavenumber in units of 2 pi / L per axis                                    */
  int store_fp32;   /* 0: populations stored fp64; 1: stored as float(f_i - w_i), arithmetic fp64 (R22)    */
  int host_staging; /* 1: workspace also holds 5 n doubles of staging so accLB_run_host can be used        */
  int device;       /* CUDA device ordinal                                                                 */
  void* stream;     /* cudaStream_t of the caller (NULL = legacy default stream)                           */
  /* the paper's two-component regime (density contrast 100, buoyant phase, time integrators) */
  double gravity[3]; /* buoyancy F^g = (rho(phi) - rho_ref) g, a force density like the others (R3, R31)
                        PAPER.md:L193, L203 ("buoyant gas phase"); single component: the uniform (1 - rho_ref) g   */
  double rho_ref;    /* reference density of F^g; the mean density gives no net force on the periodic box (R31)   */
  int phi_integrator; /* 0: forward Euler, once per LB step (R13) | 1: three-stage SSP Runge-Kutta with u frozen at
                         time t, the normal recomputed from every stage field (R32)      */
  /* moment-representation storage */
  int moment_storage; /* 1: the state is the paper's ten macroscopic fields (p*, u, a) per node instead of 27 populations
                         (160 B instead of 432 B moved per node and step; same results to rounding); single component,
                         fp64 only (two_phase = 0, store_fp32 = 0) */
  /* z-slab decomposition over several GPUs (PAPER.md:L114 halo exchange, L126 slab weak scaling) */
  int halo_z;    /* 0: the box is periodic in z (one GPU holds the whole domain).  h > 0: the box is one z-slab of a larger
                    periodic domain: its first and last h planes are HALO planes, copies of the neighbouring slabs' boundary
                    planes that the caller refreshes after every step (accLB_halo_chunks); only planes [h, nz - h) are this
                    slab's own nodes.  Needs h >= 3 for two_phase (WENO5 radius 3, R12), h >= 1 otherwise, nz >= 3 h;
                    forward Euler, population storage only (phi_integrator = 0, moment_storage = 0).                     */
  int z_origin;  /* halo_z > 0: global z coordinate of local plane 0 (may be negative: periodic), for the body force R20   */
  int nz_global; /* halo_z > 0: planes of the whole domain (the period of the body force along z)                          */
} accLB_params;

/* Bytes of device workspace accLB_create needs for this grid and these parameters; 0 on invalid arguments
 * (nx, ny, nz >= 4, nx even, nx*ny*nz < 2^31, 27*nx*ny < 2^32, tau > 0.5, two_phase: rho_l, rho_g > 0, width > 0). */
size_t accLB_workspace_bytes(int nx, int ny, int nz, const accLB_params* params);

/* Create a context on `workspace` (DEVICE pointer, caller-owned, 256-byte aligned, >= workspace_bytes).
 * Builds the body-force tables (R20) on the host with libm and uploads them.  *out is set on success. */
int accLB_create(accLB_ctx** out, int nx, int ny, int nz, const accLB_params* params, void* workspace,
                 size_t workspace_bytes);

/* Initial state (R15): f_i = f_i^eq(p*, u0) - S_i(u0, A)/2 with A from F^s + F^p + F^b, step counter := 0.
 * rho, u, phi: DEVICE pointers, caller-owned, read-only, fp64; phi may be NULL when two_phase = 0.
 * Enqueues on the stream; the inputs must stay valid until the stream reaches that point. */
int accLB_init(accLB_ctx* ctx, const double* rho, const double* u, const double* phi);

/* Advance nsteps >= 0 time steps (rows a1-a8 of DESIGN.md section 1).  Enqueues only; does not synchronise. */
int accLB_step(accLB_ctx* ctx, int nsteps);

/* Macroscopic fields of the current state: rho := p* = sum f_i, u = sum f_i c_i + A/2 (R4),
 * phi.  DEVICE pointers, caller-owned, written; any may be NULL (phi is ignored when two_phase = 0).
 * The state is unchanged.  Enqueues only. */
int accLB_moments(accLB_ctx* ctx, double* rho, double* u, double* phi);

/* Diagnostics of the current state (R21) into out[0..ACCLB_NDIAG-1] (HOST pointer, n_out >= ACCLB_NDIAG):
 *   0 KE = <rho(phi) |u|^2 / 2>      1 dissipation = <nu a:a / (2 cs^4 tau^2)>
 *   2 sum phi   3 sum p*   4..6 sum_x sum_i f_i c_i   7 max |u|   8 step count.
 * With halo_z = h > 0 the sums, means and the maximum run over the slab's own planes [h, nz - h) only.
 * Warp-shuffle + one atomic per block and quantity.  Synchronises the stream.  ACCLB_ENUMERIC if non-finite. */
int accLB_diagnostics(accLB_ctx* ctx, double* out, int n_out);

/* The same path fed from HOST buffers (what an application without device arrays calls; bench.py's e2e leg):
 * copy rho,u,phi host->device (staging), accLB_init, accLB_step(nsteps), accLB_moments, copy the three fields
 * device->host, optionally diagnostics.  Needs params.host_staging = 1.  h_* are HOST pointers (pinned memory
 * makes the copies asynchronous); outputs and h_diag (ACCLB_NDIAG doubles) may be NULL.  Synchronises. */
int accLB_run_host(accLB_ctx* ctx, const double* h_rho, const double* h_u, const double* h_phi, int nsteps,
                   double* h_rho_out, double* h_u_out, double* h_phi_out, double* h_diag);

/* Number of kernels this context has launched so far (bench.py's gpu_launches). */
long long accLB_launch_count(const accLB_ctx* ctx);

/* Per-kernel device timing.  accLB_profile(ctx, 1) makes every later launch be bracketed by two CUDA events on
 * the context's stream; accLB_profile_read synchronises the stream, adds the elapsed milliseconds and launch
 * counts per kernel kind into ms[k], count[k] for k < min(n, ACCLB_NKERNELS) (HOST pointers) and clears the
 * record.  Kinds (the names are the kernels' own, as an ncu launch list shows them): 1 k_lb (the one-node-per-thread fused
 * LB step of single-phase contexts), 3 k_init, 4 k_moments, 5 k_diagnostics (single-phase kernels, or the tiled kernel
 * k_lb_tp in its init / moments / diagnostics mode for two-phase contexts), 6 k_lb_tp (the tiled two-phase step: LB +
 * geometry + advection), 7 k_seam (advective fluxes through the faces between its tile columns), 8 k_advect (variant 1
 * and the Runge-Kutta stages), 9 k_geom_r (D lap phi - kappa div q of a Runge-Kutta stage field), 10 k_mr_step (the single-phase step on the ten
 * macroscopic fields, moment_storage = 1), 11 k_lb_tp in its Runge-Kutta stage mode (phi_integrator = 1); 0 and 2 are unused.
 * This is how bench.py measures kernel durations inside the timed region. */
#define ACCLB_NKERNELS 12
int accLB_profile(accLB_ctx* ctx, int enable);
int accLB_profile_read(accLB_ctx* ctx, double* ms, long long* count, int n);

/* Select the kernel variant of the forward-Euler two-phase step: 0 = default (k_lb_tp fused with the advection + k_seam);
 * 1 = the unfused form, u(t) and r through HBM (k_lb_tp unfused + k_advect: the path the SSP-RK3 integrator runs on),
 * kept so that bench.py / ncu can compare fused and unfused on identical inputs.  Results are
 * identical to rounding.  With phi_integrator = 1: 0 = the fused step is the first Runge-Kutta stage (it also writes u(t)) and
 * the two later stages run in the same tiled kernel without its LB half, each followed by k_seam; 1 = k_lb_tp unfused, then
 * k_advect / k_geom_r per stage.  Single-phase contexts have one path.  ACCLB_EINVAL for an unknown variant. */
int accLB_set_variant(accLB_ctx* ctx, int variant);

/* ---- z-slab decomposition ("halo regions ... exchanged between neighbouring subdomains",
 * L126 slab weak scaling).  A context created with params.halo_z = h > 0 advances a box whose first and last h planes are
 * halo planes.  One step leaves its own planes [h, nz - h) correct provided that, before the step, the halo planes hold
 * the neighbours' current state in the parts listed below; everything else in the halo planes is scratch (it is advanced
 * like the rest of the box with a periodic wrap that means nothing, and is never read by a node of [h, nz - h)).
 *   populations (stored post-collision, pulled at the next step: f_i(x, t+1) = f*_i(x - c_i, t)):
 *     low side   plane h-1: c_z >= 0 (i = 9..26; c_z = +1 streams into plane h, c_z = 0 completes the moments of plane
 *                h-1 whose velocity u enters the phi flux through the face between h-1 and h);  plane h-2: c_z = +1 only
 *                (i = 18..26; pulled by plane h-1).  Single component: plane h-1, c_z = +1 only.
 *     high side  mirrored: plane nz-h: i = 0..17, plane nz-h+1: i = 0..8.
 *   phi: all h halo planes of either side (WENO5 radius 3; curvature of plane h-1 reaches phi of plane h-3).
 * accLB_halo_chunks lists, for the CURRENT state buffers (they alternate from step to step: call it after every step), the
 * contiguous DEVICE byte ranges to send to and to receive from the two z-neighbours: out[j] for j < return value <= cap.
 *   side  -1: the neighbour that owns the planes below this slab, +1: above.    dir  0: send (read), 1: receive (written).
 * The k-th send range towards a side pairs with the k-th receive range from the opposite side of that neighbour, and has the
 * same length.  full != 0 lists every population of all h halo planes instead of the minimal set (3 x the bytes; then
 * nothing in the halo planes is scratch).  The copy itself is the caller's (NCCL send/recv, peer copies).
 * Returns the number of ranges, or a negative error (ACCLB_EINVAL: NULL, halo_z = 0, cap too small). */
typedef struct {
  void* ptr;    /* DEVICE address inside the workspace */
  size_t bytes;
  int side;     /* -1 | +1 */
  int dir;      /* 0 send | 1 receive */
} accLB_halo_chunk;
#define ACCLB_MAX_HALO_CHUNKS 16
int accLB_halo_chunks(accLB_ctx* ctx, int full, accLB_halo_chunk* out, int cap);

/* Free the context (host memory only; the workspace stays the caller's). */
int accLB_destroy(accLB_ctx* ctx);

/* Text of the last error on this thread ("" if none).  The pointer stays valid until the next call. */
const char* accLB_last_error(void);

/* ---- On-device turbulence statistics of a velocity field.  Context-free:
 * u is a DEVICE pointer to [3][nz][ny][nx] fp64 (e.g. the u of accLB_moments), results go to HOST pointers, `scratch` is a
 * small caller-owned DEVICE block (8-byte aligned) for the accumulators; the calls synchronise `stream`.
 *
 * accLB_stats_increments: longitudinal structure functions, for each separation r[j] >= 0 (HOST array):
 *   out[3 j + p - 2] = S_p(r_j) = < (u_a(x + r e_a) - u_a(x))^p >, p = 2, 3, 4, averaged over all nodes and the three
 *   axes a (periodic).  The longitudinal gradient of PAPER.md:L183, taken as the central difference, has the moments
 *   S_p(2) / 2^p: skewness S_3(2) / S_2(2)^{3/2}, flatness S_4(2) / S_2(2)^2.  scratch >= 3 nr doubles.
 * accLB_stats_pdf: histogram of d / scale, d the same increments at separation r (r = 2, scale = 2 rms: the gradient PDF of
 *   PAPER.md Fig. 3a; any r: the increment PDFs of Fig. 6), nbins <= 1024 equal bins on [lo, hi); values outside go to
 *   the first / last bin.  counts: HOST, nbins entries, sum = 3 nx ny nz.  scratch >= nbins 8-byte counters.
 * accLB_stats_spectrum: shell sums of a real-to-complex transform (Fig. 2, 5): uhat is a DEVICE pointer to
 *   [ncomp][nz][ny][nx/2 + 1] complex fp64 (re, im interleaved), the UNNORMALISED transform of ncomp real fields (the FFT
 *   is the caller's library call); E[k] = sum over the modes with round(|k|) = k of |uhat|^2 / (2 N^2), the conjugate
 *   half counted, k = 0 .. nshell - 1, so that sum_k E[k] = < f.f > / 2 when nshell covers all modes.  scratch >= nshell
 *   doubles. */
int accLB_stats_increments(const double* u, int nx, int ny, int nz, const int* r, int nr, double* out, void* scratch,
                           size_t scratch_bytes, int device, void* stream);
int accLB_stats_pdf(const double* u, int nx, int ny, int nz, int r, double scale, double lo, double hi, int nbins,
                    unsigned long long* counts, void* scratch, size_t scratch_bytes, int device, void* stream);
int accLB_stats_spectrum(const double* uhat, int nx, int ny, int nz, int ncomp, int nshell, double* E, void* scratch,
                         size_t scratch_bytes, int device, void* stream);

/* ---- The same structure functions for callers that cannot allocate device memory (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): accLB_stats_increments without the caller's scratch block.  The
 * accumulators (3 nr doubles) live in ONE fixed array of device memory inside the library (file scope, 256-byte aligned,
 * 3 * ACCLB_STATS_STATIC_MAX_NR doubles = 1536 bytes; every GPU that loads the library holds it until the process exits).
 * The call allocates nothing: no cudaMalloc / cudaFree, no allocating library routine; it zeroes the accumulators it uses,
 * launches the same kernel as accLB_stats_increments, copies the 3 nr sums to `out` (HOST) and synchronises `stream`.
 *   u, r, nr, out, device, stream: as for accLB_stats_increments.  nr > ACCLB_STATS_STATIC_MAX_NR -> ACCLB_EINVAL.
 * ALL calls on a device share the array, which keeps the last call's contents: two calls that overlap on the GPU (different
 * streams, or different host threads) race on it and give wrong sums -- serialise them, or use accLB_stats_increments with
 * one scratch block per caller. */
#define ACCLB_STATS_STATIC_MAX_NR 64
int accLB_stats_increments_static(const double* u, int nx, int ny, int nz, const int* r, int nr, double* out, int device,
                                  void* stream);

#ifdef __cplusplus
}
#endif
#endif /* ACCLB_H */
