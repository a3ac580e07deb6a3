/*
 * mm.h — C ABI of the B200-native LLG hot path (arxiv 2406.16064, "MicroMagnetic.jl").
 *
 * One handle = one finite-difference micromagnetic problem on a regular nx*ny*nz mesh
 * ("FDMesh", "cell-based" Ms).  The calls below are the hot path of
 * one Landau-Lifshitz-Gilbert time step: effective field (Eq. 1; demag Eq. 8
 * PAPER.md:138-140 as a zero-padded FFT convolution; exchange Eq. 5; DMI Eq. 15
 * PAPER.md:173-175; uniaxial anisotropy Eq. 32 PAPER.md:269 in its continuum reading; Zeeman
 * Eq. 35), the LL torque (Eq. 37) and a Dormand-Prince / RK4 step with
 * projection onto |m| = 1.  Every step of the path runs in the library's
 * CUDA kernels (sm_100a); there is no CPU fallback.
 *
 * Conventions
 *  - Every function returns an mm_status (0 = MM_OK) unless stated; no exception crosses the ABI.
 *  - Pointers named dev_* are DEVICE pointers on the handle's device, in the handle's precision
 *    (float for MM_F32, double for MM_F64), owned by the caller.  Pointers named host_* are HOST
 *    pointers.  Out-parameters (int*, double*, long*) are HOST pointers and may be NULL.
 *  - Layout: x fastest, cell index idx = i + nx*(j + ny*k); vector fields are SoA: component c of
 *    cell idx is at [c*N + idx], N = nx*ny*nz, c in {x, y, z}.  Ms is N reals; Ms = 0 marks vacuum.
 *  - Units: SI.  m dimensionless unit vectors; H in A/m; Ms in A/m; A in J/m; D in J/m^2; Ku in
 *    J/m^3; gamma in m/(A s); time in s; cell edges in m.  mu0 = 4 pi 1e-7.
 *  - A neighbour outside the mesh or with Ms = 0 is absent (free boundary).  Cells with Ms = 0 get
 *    H = 0 and dm/dt = 0, and are never touched by the integrators.
 *  - All work is enqueued on the CUDA stream given to mm_create and is asynchronous with respect
 *    to the host unless a non-NULL host out-parameter (or a host_* buffer) forces a
 *    synchronisation of that stream.
 *  - Meshes: any nx, ny, nz >= 1 (nz = 1: thin film).  The FFT passes are radix-2: a size that is not a power of two
 *    is embedded in the next power of two with vacuum cells (the caller's arrays keep their own nx*ny*nz layout; the
 *    library packs / unpacks at every call, two small kernels); powers of two take the direct path.  With demag
 *    enabled the padded mesh needs nx >= 4, ny >= 2 and the per-CTA shared-memory tiles must fit (see DESIGN.md
 *    "Limits"); otherwise mm_init_demag returns MM_ERR_UNSUPPORTED.
 */
#ifndef MM_H
#define MM_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mm_sim mm_sim;  /* opaque; created/destroyed only by the library */

typedef enum { MM_F32 = 0, MM_F64 = 1 } mm_prec;
typedef enum {
    MM_OK = 0,
    MM_ERR_ARG = -1,          /* bad argument (NULL, non-positive size, zero axis, ...)        */
    MM_ERR_UNSUPPORTED = -2,  /* mesh shape outside the supported set                           */
    MM_ERR_STATE = -3,        /* call order: e.g. demag enabled but mm_init_demag not called,   */
                              /* or workspace not set                                           */
    MM_ERR_CUDA = -4,         /* a CUDA runtime call or kernel launch failed                    */
    MM_ERR_NOMEM = -5,        /* workspace too small / allocation failed                        */
    MM_ERR_NAN = -6,          /* non-finite error norm met in mm_step / mm_relax                */
    MM_ERR_INTERNAL = -7      /* a self-check of the library failed (e.g. K^ not real at setup)   */
} mm_status;
/* DMI vectors e_ij for the neighbours {-x,+x,-y,+y,-z,+z}: bulk r^_ij; interfacial z^ x r^_ij =
 * {-y^,+y^,+x^,-x^,0,0}; D2d {+x^,-x^,-y^,+y^,0,0} (Eq. 14). */
typedef enum { MM_DMI_NONE = 0, MM_DMI_BULK = 1, MM_DMI_INTERFACIAL = 2, MM_DMI_D2D = 3 } mm_dmi_kind;
/* MM_CAYLEY_RK4: classical RK4 on omega of the Cayley transform (Eq. 43-49), omega restarted at 0
 * every step, m <- Q(omega) m; fixed step, no projection (Q is a rotation).  In fp32 the rounding of Q m lets |m| drift
 * like a random walk, about 1e-7 sqrt(steps) (measured 2e4 steps: tests/test_gpu_torques.py); callers running millions
 * of fp32 Cayley steps should renormalise m themselves now and then. */
typedef enum { MM_RK4 = 0, MM_DOPRI5 = 1, MM_CAYLEY_RK4 = 2 } mm_integrator;

/* Create a problem on `device`, all later work on `cuda_stream` (a cudaStream_t; NULL = default
 * stream).  dx, dy, dz: cell edges in metres.  Defaults: Ms = 0 everywhere, A = D = Ku = 0, axis =
 * z, H_ext = 0, alpha = 0.5, gamma = 2.211e5, integrator = MM_DOPRI5, demag enabled. */
int mm_create(mm_sim** out, int nx, int ny, int nz, double dx, double dy, double dz,
              mm_prec prec, int device, void* cuda_stream);
int mm_destroy(mm_sim* sim);

/* Persistent device memory the library needs (cached tensor spectrum K^, FFT spectra, RK stage
 * vectors, Ms).  The CALLER allocates it (e.g. torch.empty) and keeps it alive until mm_destroy;
 * the library only carves it up.  Must be called before mm_set_Ms / mm_init_demag / any compute.
 * mm_init_demag builds the padded tensor inside this workspace (in slots that hold nothing before the first
 * evaluation); it cudaMallocs only the real-space tensor (6N doubles) and small tables, and frees them on
 * every exit path.
 * Alignment: every device pointer handed to the library (m, H, dm/dt, Ms) must be 16-byte aligned (the
 * kernels use 16-byte vector accesses); torch allocations are, offset views of them may not be. */
size_t mm_workspace_bytes(const mm_sim* sim);
int mm_set_workspace(mm_sim* sim, void* dev_ptr, size_t bytes);   /* dev_ptr 256-byte aligned */

/* Material / run parameters (Listing 2 names). */
int mm_set_Ms_uniform(mm_sim* sim, double Ms);
int mm_set_Ms(mm_sim* sim, const void* dev_Ms);                   /* N reals, copied            */
int mm_set_A(mm_sim* sim, double A);
int mm_set_D(mm_sim* sim, double D, mm_dmi_kind kind);
int mm_set_Ku(mm_sim* sim, double Ku);
int mm_set_axis(mm_sim* sim, double ux, double uy, double uz);    /* normalised inside; 0 => ARG */
int mm_set_H_ext(mm_sim* sim, double hx, double hy, double hz);
/* Cell-based material constants (PAPER.md:66 "cell-based", :120, :175): dev_A / dev_D hold N reals in the handle's
 * precision, copied into the workspace.  The bond values are the harmonic means A_ij = 2 A_i A_j / (A_i + A_j)
 * and D_ij = 2 D_i D_j / (D_i + D_j), 0 when both vanish.  While set they replace the
 * uniform mm_set_A / mm_set_D value; NULL (or a later mm_set_A / mm_set_D) switches back.  `kind` takes effect only
 * when dev_D is non-NULL and the copy succeeded: mm_set_D_cell(sim, NULL, kind) keeps the kind of the last mm_set_D,
 * and a call that returns an error changes nothing.  Call after mm_set_workspace. */
int mm_set_A_cell(mm_sim* sim, const void* dev_A);
int mm_set_D_cell(mm_sim* sim, const void* dev_D, mm_dmi_kind kind);
/* Cubic anisotropy, Eq. 33 in its continuum reading (R6): energy density
 * Kc (mx^4 + my^4 + mz^4), crystal axes = mesh axes, H = -(4 Kc / (mu0 Ms)) (mx^3, my^3, mz^3).  mm_energy reports it
 * inside the anisotropy term. */
int mm_set_Kc(mm_sim* sim, double Kc);
/* Per-cell external field (Eq. 35 with H_i): dev_H holds 3N reals (SoA, A/m), copied; NULL
 * switches back to the uniform mm_set_H_ext value. */
int mm_set_H_ext_cell(mm_sim* sim, const void* dev_H);
/* Zhang-Li spin-transfer torque: dm/dt += f_stt x m, f_stt = [(beta - alpha) tau + (1 + alpha beta)
 * m x tau] / (1 + alpha^2), tau = (u . grad) m by central differences (a missing neighbour is replaced
 * by the cell itself).  u in m/s (Eq. 39), uniform; (0,0,0) switches the term off.  Sign convention of Eq. 44 / Eq. 54
 * (a head-to-head wall moves with -(1 + alpha beta) u / (1 + alpha^2)); Eq. 38 as printed has u -> -u (R17). */
int mm_set_zhang_li(mm_sim* sim, double ux, double uy, double uz, double beta);
/* Time profile of that current: u(t) = u exp(-b t) cos(w t) (the pulse of PAPER.md:444; Eq. 54 holds for any u(t)),
 * evaluated at every RK stage's own time t + c dt on the device.  b = w = 0 (the default): constant current. */
int mm_set_zhang_li_pulse(mm_sim* sim, double b, double w);
/* Slonczewski / spin-orbit torque, Eq. 40: -a_J m x (m x p) - b_J m x p added to the Gilbert
 * equation; a_J, b_J in 1/s, p normalised inside (zero p with non-zero a_J or b_J => MM_ERR_ARG). */
int mm_set_slonczewski(mm_sim* sim, double a_J, double b_J, double px, double py, double pz);
/* Thermal field, Eq. 41-42: xi = eta sqrt(2 alpha kB T / (mu0 Ms gamma V dt)) added to H_eff during
 * mm_step / mm_relax / mm_run_until / mm_run_host, one Gaussian vector per cell and step attempt (held over the stages),
 * eta from Philox4x32-10 + Box-Muller keyed by (seed, attempt counter, cell index) (R18).  Resets the
 * attempt counter.  T = 0 switches it off.  mm_effective_field / mm_llg_rhs never include it.  Needs the workspace.
 * Fixed steps only: while T > 0, mm_step / mm_run_host with tol > 0 under MM_DOPRI5, mm_relax and mm_run_until return
 * MM_ERR_UNSUPPORTED — xi depends on dt (Eq. 42) and a rejected attempt would throw its noise away and redraw, which
 * biases the noise the accepted steps see; the paper gives no rule for it, so the library refuses rather than guess. */
int mm_set_temperature(mm_sim* sim, double T_kelvin, unsigned long long seed);
/* The thermal field a step of size dt with attempt counter `step` would use: 3N reals to dev_out (parity tests). */
int mm_thermal_field(mm_sim* sim, double dt, unsigned long long step, void* dev_out);
int mm_set_alpha(mm_sim* sim, double alpha);
int mm_set_gamma(mm_sim* sim, double gamma);
int mm_set_integrator(mm_sim* sim, mm_integrator integ);
int mm_set_demag(mm_sim* sim, int on);                            /* 0/1; default 1             */

/* Build and cache the spectrum of the demag tensor (depends on mesh and cell size
 * only).  Tensor in fp64 (near field: closed forms of ref [20] in __float128 on the host; far
 * field: Gauss-Legendre quadrature of the defining dipole integral in fp64 on the device), its
 * FFT in fp64, rounded once to the handle's precision.  Synchronous. */
int mm_init_demag(mm_sim* sim);

/* H_eff(m) — Eq. 1 with all enabled terms.  dev_m, dev_H: 3N reals each. */
int mm_effective_field(mm_sim* sim, const void* dev_m, void* dev_H);
/* dm/dt — Eq. 37.  dev_dmdt: 3N reals, 1/s. */
int mm_llg_rhs(mm_sim* sim, const void* dev_m, void* dev_dmdt);

/* One step of the selected integrator, m updated in place on acceptance, time advanced.
 * tol <= 0: fixed step, always accepted.  DOPRI5 (R8): err = max_i |dt sum_j e_j k_j|,
 * accept iff err <= tol, dt_next = dt * clamp(0.9 (tol/err)^(1/5), 0.2, 5).  7 RHS evaluations per
 * step (no FSAL).  RK4: 4 RHS evaluations, err = 0.  max_dmdt = max_i |k_1,i|.
 * If all four out-pointers are NULL the call does not synchronise. */
int mm_step(mm_sim* sim, void* dev_m, double dt, double tol,
            int* accepted, double* err, double* dt_next, double* max_dmdt);

/* Adaptive steps (DOPRI5) from dt0 until max|dm/dt| < stop_dmdt (rad/s) or max_steps steps
 * (accepted + rejected).  dt0 (the first trial step, seconds) is an addition to SURVEY.md 8(b)'s
 * signature: the paper gives no rule for it and the caller knows the time scale.
 * The step controller runs on the device; the host reads the device state back every 16 steps,
 * kernels enqueued after the stop condition return at once. */
int mm_relax(mm_sim* sim, void* dev_m, double tol, double stop_dmdt, long max_steps, double dt0,
             long* steps_done, double* max_dmdt);

/* Energy minimisation by steepest descent with Barzilai-Borwein steps (§VI).  Per iteration k:
 * f_k = m x H_eff(m_k), g_k = m x (m x H_eff(m_k)); the modulus-preserving update of Eq. 51,
 * (1 + tau^2 f_k^2/4) m_{k+1} = (1 - tau^2 f_k^2/4) m_k - tau g_k, per cell; step size by Eq. 52 with
 * s = m_k - m_{k-1}, y = g_k - g_{k-1}: tau^1 = sum s.s / sum s.y on odd k, tau^2 = sum s.y / sum y.y on even k
 * (sums over cells with Ms > 0, fp64, fixed order).  Readings where the paper is silent (R16): tau0 (m/A)
 * for the first update, |tau| clamped to [tau_min, tau_max], a vanishing / non-finite quotient falls back to tau0.
 * Stops before the update when max_i |g_k,i| < stop_torque (A/m) or after max_steps updates.  dev_m (3N reals) is
 * updated in place; no projection is applied (Eq. 50 keeps |m|).  Out-pointers may be NULL.  Synchronous. */
int mm_minimize(mm_sim* sim, void* dev_m, double tau0, double tau_min, double tau_max, double stop_torque, long max_steps,
                long* steps_done, double* max_torque, double* tau_last);

/* Advance by adaptive DOPRI5 steps until exactly t_end (last step clipped). */
int mm_run_until(mm_sim* sim, void* dev_m, double t_end, double tol, double dt0, long max_steps,
                 long* steps_done);

/* End-to-end convenience with HOST buffers: copies host_m (3N reals) to the device, takes
 * nsteps fixed-dt steps (tol <= 0) or adaptive attempts (tol > 0), copies m back.  Synchronous. */
int mm_run_host(mm_sim* sim, void* host_m, int nsteps, double dt, double tol);
/* Same for one RHS evaluation: host_m in, host_dmdt out. */
int mm_llg_rhs_host(mm_sim* sim, const void* host_m, void* host_dmdt);

double mm_time(mm_sim* sim);                                      /* synchronises the stream to read the device clock */
int mm_set_time(mm_sim* sim, double t);

/* Diagnostics, off the hot path (synchronous). */
int mm_average_m(mm_sim* sim, const void* dev_m, double out3[3]);   /* mean over cells with Ms>0 */
/* <m> for callers that cannot provide device memory.  mm_average_m (above) needs a handle and its workspace, a buffer
 * of hundreds of megabytes that the caller has to allocate.  This call needs neither: the partial sums go to an array
 * that is built into the library (256 B + 512 KiB of every GPU that loads libmm.so, held until the process exits), and
 * the call allocates and frees nothing, on the host or on the device.  It is meant for code that wants to watch <m> but
 * is in no position to allocate: a logging hook inside an application whose memory pool already owns all of HBM (a
 * plain cudaMalloc fails there), code inside a latency-critical loop that cannot afford the device-wide wait of
 * cudaMalloc / cudaFree, or a plug-in that is handed two arrays and a stream and nothing else.
 *   device, cuda_stream : the device the arrays live on (made current, like every mm_* call does) and the stream the
 *                         work is enqueued on (a cudaStream_t; NULL = default stream).  Asynchronous: nothing waits.
 *   prec, ncells        : element type of dev_m / dev_Ms; number of cells N, 1 <= N <= MM_STATIC_MAX_CELLS.  A larger N
 *                         returns MM_ERR_UNSUPPORTED (message in mm_static_last_error) and enqueues nothing.
 *   dev_m, dev_Ms       : 3N and N reals, SoA as everywhere in this header, read only; natural alignment suffices.
 *   dev_out3            : 3 doubles on the device, written by the kernel: the mean of m over cells with Ms != 0 (0 if
 *                         there is none) — the same number mm_average_m returns, both sum in fp64.
 * Sharing: there is ONE built-in array per device.  Calls on the same stream are safe.  Two calls that can run on the
 * GPU at the same time (different streams or host threads) overwrite each other's partial sums: both results are then
 * undefined; order them yourself.  The array keeps the previous call's contents; the call clears the one word that
 * must start at zero (its block counter) on `cuda_stream` before the kernel, the rest is overwritten before it is read.
 * First call on a device: looks up the array's device address, which makes the driver load the library's device code
 * there if it has not yet.  Make that first call once per device during start-up, before any stream capture begins
 * and before the latency-critical part of the program; later calls enqueue one 256-byte memset and one kernel. */
#define MM_STATIC_MAX_CELLS (1L << 26)   /* 67 108 864 cells, e.g. 8192 x 8192 x 1 or 1024 x 1024 x 64 */
int mm_average_m_static(int device, void* cuda_stream, mm_prec prec, long ncells, const void* dev_m, const void* dev_Ms,
                        double* dev_out3);
/* Message of the last mm_average_m_static failure on the calling host thread ("" after a success); static storage. */
const char* mm_static_last_error(void);
/* E = -mu0 V sum_i Ms_i m_i.(H_d/2 + H_ex/2 + H_dmi/2 + H_an/2 + H_ext); terms in that order. */
int mm_energy(mm_sim* sim, const void* dev_m, double* E_total, double E_terms[5]);
/* Real-space tensor component (0..5 = xx,yy,zz,xy,xz,yz) at offsets i,j,k >= 0: N doubles (fp64
 * regardless of precision) to dev_out.  Valid after mm_init_demag. */
int mm_get_demag_kernel(mm_sim* sim, int comp, void* dev_out);
/* Per-kernel timing for roofline accounting (bench.py).  While on, the library brackets each hot-path
 * kernel with CUDA events on the handle's stream; mm_get_profile synchronises the stream, sums the
 * elapsed milliseconds and launch counts per kernel class since the last call — [0] pass A
 * fwd_xz, [1] pass B y_conv, [2] pass C inv_zx, [3] fused local-field/torque/RK-stage kernel —
 * and clears the record.  Off by default (no events are recorded).  on = 1: all four classes; any other
 * value is a bit mask (bit c+1 = class c, e.g. 4 = pass B only), so that a benchmark can bracket only its dominant kernel and keep
 * the event overhead (two stream operations per kernel) out of the rest of the step. */
int mm_set_profiling(mm_sim* sim, int on);
int mm_get_profile(mm_sim* sim, double ms_out[4], long count_out[4]);
/* Step statistics, kept by the device-side controller: step attempts accepted and rejected by mm_step / mm_relax /
 * mm_run_until / mm_run_host since mm_set_workspace, and the RHS evaluations (Eq. 37) those attempts made (7 per DOPRI5
 * attempt, 4 per RK4 / Cayley-RK4 attempt; mm_effective_field, mm_llg_rhs and mm_minimize are not counted).  Attempts
 * enqueued after a stop condition was met do no work and are not counted.  Out-pointers are HOST pointers and may be
 * NULL.  Synchronises the stream. */
int mm_get_stats(mm_sim* sim, long* accepted, long* rejected, long* rhs_evals);
/* Number of kernel launches issued by this handle so far (for bench accounting). */
long mm_launch_count(const mm_sim* sim);
const char* mm_last_error(const mm_sim* sim);
const char* mm_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MM_H */
