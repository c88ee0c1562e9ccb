/*
 * kx.h -- C ABI of libkx: the discretized 2->2 elastic self-collision operator C[f] of KineticXGPU
 * (arxiv/paper_2607_00755) as hand-written CUDA for sm_100a (NVIDIA B200).
 *
 * What the library computes (citations are PAPER.md line numbers; readings D1-D13 are in DESIGN.md):
 *   kinematics        E_i = sqrt(p_i^2+m^2), K_i = E_i-m, h_i = p_i^2 dp_i          eq. B.1
 *   index map         E_j~ = E_n+E_m-E_i, bracket j_L and weight omega_R            eq. 4.4, B.19
 *   kernel tensor     W_inm = dp_n dp_m F_inm / (2 E_i g_chi)                        eq. 4.7, B.15-B.17
 *   operator          C_i = sum_{n,m} W_inm (f_n f_m - f_i f_j~)                     eq. 4.6 with eq. 2.6
 *                     or with the quantum factors of eq. 4.3 for KX_STAT_BOSE / KX_STAT_FERMI
 *   interpolation     f_j~ = exp(w_L ln f_L + w_R ln f_R)  (LOG)  or  w_L f_L + w_R f_R (LINEAR)   eq. B.20
 *   projection        C^proj = C^raw - xi_i (alpha + beta E_i)                       App. C, eq. C.2-C.8
 *   moments           n = g/(2 pi^2) sum h f, rho = g/(2 pi^2) sum h E f             eq. B.2
 *   time stepping     df/dtau = kappa_b R(tau) C^proj[f; m(tau)] + sum_s amp_s G_s   eq. 4.9
 *
 * Conventions
 *   - Every function returns kx_status_t (KX_OK = 0).  No exceptions, no abort(), no state shared between handles.
 *     kx_last_error(h) returns a handle-owned, NUL-terminated description of the last failure; kx_last_error(NULL)
 *     returns the calling thread's last kx_build failure (thread-local: there is no handle to own it).
 *   - Pointers are marked HOST or DEVICE.  DEVICE pointers are caller-owned allocations on the
 *     handle's device (e.g. torch.Tensor.data_ptr()), 16-byte aligned, row-major [B,N] fp64.
 *     HOST arrays are read during the call and may be freed afterwards.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  kx_collide*,
 *     kx_moments and kx_set_mass only enqueue work on it and return without synchronising, with two
 *     exceptions: (1) the first call with a larger batch B than seen before grows the handle's workspace
 *     (cudaMalloc, implicit sync) -- kx_reserve(h, B) does that ahead of time; (2) on a KX_STORE_TILED handle
 *     the first kx_collide* / kx_evolve* after kx_set_mass (or after a mass-schedule kx_evolve) rebuilds the
 *     tiled operand, which synchronises the stream and may reallocate it; the first kx_set_mass itself
 *     synchronises and reallocates the row storage to N^2 (N+1)/2 entries (every triple may be kept at
 *     another mass).  kx_build, kx_evolve, kx_evolve_adaptive, kx_collide_host and kx_tensor_export
 *     synchronise the stream before returning.
 *   - One operator evaluation is one cooperative kernel launch (all of its CTAs are resident at once and
 *     meet at a grid barrier); run other work on the same device in the same stream or expect it to
 *     serialise with the evaluation.
 *   - The handle owns the kernel tensor and all workspaces.  One host thread at a time per handle.
 *   - There is no CPU fallback: every entry point fails with KX_ERR_CUDA when no sm_100 device
 *     is usable.
 */
#ifndef KX_H_
#define KX_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct kx_handle_s* kx_handle_t;

typedef enum {
    KX_OK = 0,
    KX_ERR_INVALID_ARG = 1,   /* null pointer, N<4, non-monotone grid, dp<=0, B<1, misaligned pointer */
    KX_ERR_ALLOC = 2,         /* host or device allocation failed */
    KX_ERR_CUDA = 3,          /* CUDA runtime error (message in kx_last_error) */
    KX_ERR_UNSUPPORTED = 4,   /* option not implemented (fp32 with quantum statistics, LINEAR with statistics); N > 1024 (n, m, j_L
                                 are packed 10 bits each) */
    KX_ERR_NONFINITE = 5      /* kx_evolve produced a NaN/Inf in f */
} kx_status_t;

/* interpolation of f at the off-grid fourth momentum (reading D7) */
#define KX_INTERP_LOG     0   /* eq. B.20 at eta=0: f_j~ = exp(w_L y_L + w_R y_R), y = ln max(f, f_floor) (default) */
#define KX_INTERP_LINEAR  1   /* f_j~ = w_L f_L + w_R f_R (operator exactly bilinear) */
/* storage of the kernel tensor */
#define KX_STORE_SYM_ROWS 0   /* symmetry-reduced (n<=m, W_inm+W_imn), structural zeros dropped, row-compressed;
                                 evaluated by the streaming kernel, one exp per (entry, member) in LOG mode */
#define KX_STORE_TILED    1   /* default: SYM_ROWS plus the 16-row tiled operand of the FP64 tensor-core (DMMA)
                                 contraction: gain as (n<=m) x members GEMM, LOG loss through the Chebyshev moments
                                 of each (i, bracket) bucket; members with a bracket whose
                                 interpolation error bound exceeds 1e-15 max f fall back to the streaming kernel */
/* precision */
#define KX_FP64 0
#define KX_FP32 1             /* optional: the contraction (a4-a5) in single precision on the streaming kernel (the paper's GPU timings
                                 are fp32); interface arrays stay fp64; error <= 1e-4 of max |gain| (BASELINE.json);
                                 classical statistics only (else KX_ERR_UNSUPPORTED); forces KX_STORE_SYM_ROWS */
/* exp used by the LOG loss term */
#define KX_EXP_TABLE 0        /* 256-entry table x degree-4 polynomial of the remainder, <= 2 ulp (default) */
#define KX_EXP_LIBM  1        /* CUDA math library exp2() */
/* quantum statistics of the species (eq. 4.3): Lambda_inm = f_n f_m (1+eta f_i)(1+eta f_j~)
 * - f_i f_j~ (1+eta f_n)(1+eta f_m), off-grid occupation through y = ln(f/(1+eta f)) (eq. B.20).
 * eta != 0 needs KX_INTERP_LOG and is evaluated by the exact streaming kernel (the operator is no longer bilinear);
 * Fermi-Dirac needs 0 <= f < 1. */
#define KX_STAT_CLASSICAL 0   /* Maxwell-Boltzmann, the dilute limit of eq. 2.6 (default) */
#define KX_STAT_BOSE      1
#define KX_STAT_FERMI   (-1)
/* flags of kx_collide / kx_evolve */
#define KX_PROJECT 1u         /* apply the two-moment projection of App. C */
#define KX_DIAG    2u         /* kx_evolve: fill ctl->diag */
/* integrators of kx_evolve (fixed step) */
#define KX_EULER 0
#define KX_HEUN  1
#define KX_RK4   2

/* Momentum grid (HOST): p ascending and > 0, dp > 0 (bin widths / quadrature weights, reading D1). eq. 4.5 */
typedef struct { int32_t n; const double* p; const double* dp; } kx_grid_t;
/* Species: mass m >= 0 and internal degrees of freedom g_chi > 0 (eq. 4.2) */
typedef struct { double m; double g_chi; } kx_species_t;
/* |M|^2 = M2_0 (m_med <= 0: contact, eq. B.17) or M2_0 / (1 + (-t)/m_med^2)^2, t = (p_i-p_n)^2 (reading D5) */
typedef struct { double M2_0; double m_med; } kx_msq_t;
/* Options; pass NULL for the defaults {LOG, TILED, FP64, EXP_TABLE, 0, 0, 0, 0, 1e-300, 1e-12} */
typedef struct {
    int32_t interp;      /* KX_INTERP_*  */
    int32_t storage;     /* KX_STORE_*   */
    int32_t precision;   /* KX_FP64 | KX_FP32 */
    int32_t exp_impl;    /* KX_EXP_*     */
    int32_t loss_nodes;  /* KX_STORE_TILED + LOG: Chebyshev nodes per bracket, 8|16|24|32; 0 = default (24) */
    int32_t statistics;  /* KX_STAT_*: eta = 0 | +1 | -1 */
    int32_t n_mu;        /* 0 (default): analytic reduced kernel, eq. B.17 / reading D5.  > 0: the numerical angular kernel
                            F_inm of eq. B.4-B.12 with n_mu Gauss-Legendre nodes in mu = cos(p_i, p_n),
                            |M|^2 evaluated at t(mu) (O(n_mu N^3) build); n_mu <= 4096 */
    int32_t reserved;    /* must be 0 */
    double  f_floor;     /* y = ln max(f, f_floor), reading D8; must be >= 1e-300 and > 0 */
    double  eps_supp;    /* support threshold of eq. C.4, reading D9 */
} kx_opts_t;

/* a1-a3: build kinematics, the energy-conserving index map and the kernel tensor ON THE DEVICE.
 * `device` is the CUDA ordinal.  Synchronises `stream`.  *out is NULL on failure. */
kx_status_t kx_build(const kx_grid_t* grid, const kx_species_t* sp, const kx_msq_t* msq,
                     const kx_opts_t* opts, int device, void* stream, kx_handle_t* out);

/* Re-run a1-a3 for a new kinematic mass (p_i = q_i/a changes with time; reading D12).
 * Asynchronous: the new number of non-zeros stays on the device (kx_info synchronises to read it). */
kx_status_t kx_set_mass(kx_handle_t h, double m, void* stream);

/* a4-a7: C[b,i] = sum_{n,m} W_inm (f_n f_m - f_i f_j~) for B distributions (eq. 4.6).
 * f, C: DEVICE [B,N].  flags: 0 = raw operator, KX_PROJECT = App. C projection applied.
 * In place (C == f) is not allowed. */
kx_status_t kx_collide(kx_handle_t h, const double* f, double* C, int32_t B, uint32_t flags, void* stream);

/* a4, a5 separately: gain[b,i] = sum W f_n f_m, loss[b,i] = f_i sum W f_j~ (DEVICE [B,N]; either may be NULL);
 * with statistics: gain = sum W f_n f_m (1+eta f_i)(1+eta f_j~), loss = f_i sum W f_j~ (1+eta f_n)(1+eta f_m). */
kx_status_t kx_collide_parts(kx_handle_t h, const double* f, double* gain, double* loss, int32_t B, void* stream);

/* General form: any of C, gain, loss, diag may be NULL.  diag: DEVICE [B,4] = eps_N, eps_E (eq. C.1,
 * PAPER.md:415, of the raw operator) and R_N, R_E (eq. C.9; zero unless KX_PROJECT). */
kx_status_t kx_collide_ex(kx_handle_t h, const double* f, double* C, double* gain, double* loss,
                          double* diag, int32_t B, uint32_t flags, void* stream);

/* Same operator with HOST buffers f[B,N] -> C[B,N]: host->device copy of f, kx_collide, the result back to the host,
 * on `stream`, then synchronises.  Pinned host memory makes the copy of f asynchronous; a pinned (device-mapped, 16-byte
 * aligned) C_host is written by the evaluation kernel itself (no separate device->host copy: about 10 us less per call);
 * a pageable C_host goes through the handle's staging buffer and a cudaMemcpyAsync. */
kx_status_t kx_collide_host(kx_handle_t h, const double* f_host, double* C_host, int32_t B,
                            uint32_t flags, void* stream);

/* The same operator (a4-a7, C only) through an entry point that ALLOCATES NOTHING: no cudaMalloc / cudaFree / allocating
 * library routine, on any call (every other evaluation call may grow the handle's workspace on its first call with a larger
 * batch).  For callers that cannot allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid it.
 * A variant of the fused exact streaming kernel evaluates the handle's row storage (any storage mode; classical statistics,
 * fp64, else KX_ERR_UNSUPPORTED) with its scratch -- per-task partial sums, task table, grid-barrier words -- in a file-scope
 * static __device__ array of about 2 MiB that every GPU loading the library holds until exit.
 * Limit: (tasks x B) <= 131072 pairs of partial sums, tasks <= nnz / chunk + N with chunk = 4096 entries doubled up to 65536
 * until it fits (BASELINE config 3, N = 256: B <= 81 at chunk 4096, more at larger chunks; config 4, N = 512: B <= 110); beyond
 * that KX_ERR_UNSUPPORTED with a message naming the limit -- nothing is launched.
 * All calls share the array and it keeps the last call's contents (what must start at zero is cleared by every call): calls
 * that OVERLAP on one GPU (two streams, two host threads, two handles) race on it -- serialise them.  One cooperative launch
 * plus a one-CTA set-up kernel; asynchronous on `stream`.  Results equal kx_collide's up to the order of the partial sums. */
kx_status_t kx_collide_static(kx_handle_t h, const double* f, double* C, int32_t B, uint32_t flags, void* stream);

/* a9: moments of eq. B.2.  f: DEVICE [B,N]; n, rho, p1 = <p>, p2 = <p^2>: DEVICE [B], any may be NULL. */
kx_status_t kx_moments(kx_handle_t h, const double* f, int32_t B,
                       double* n, double* rho, double* p1, double* p2, void* stream);

/* Source terms of eq. 4.1/4.9: sum_s amp[s,k] G[s,i] during step k (constant over the step's stages, D11). */
typedef struct {
    int32_t nsrc;          /* 0..8 */
    const double* G;       /* DEVICE [nsrc,N] source shapes */
    const double* amp;     /* HOST [nsrc,S] rate of source s during step k, per unit tau */
} kx_source_t;

typedef struct {
    int32_t method;        /* KX_EULER | KX_HEUN | KX_RK4 */
    int32_t S;             /* number of steps */
    const double* tau;     /* HOST [S+1] nodes of the integration variable (t, or u = ln a, eq. 4.9) */
    const double* rate;    /* HOST [2S+1] multiplier R at nodes and midpoints (1/H, eq. 4.9); NULL => 1 */
    const double* mass;    /* HOST [2S+1] kinematic mass at nodes and midpoints; NULL => static tensor.
                              When given, a1-a3 are re-evaluated at every stage (reading D12). */
    const double* kappa;   /* HOST [B] per-member coupling multiplier; NULL => 1 */
    uint32_t flags;        /* KX_PROJECT | KX_DIAG */
    double* diag;          /* DEVICE [S,B,6]: eps_N, eps_E, R_N, R_E of each step's first stage, then
                              n, rho after the step (with the end-of-step mass); or NULL */
} kx_evolve_t;

/* a8: S fixed steps of df/dtau = kappa_b R C[f; m] + sources, every stage = contraction + projection +
 * fused Runge-Kutta update on the device.  f: DEVICE [B,N], in/out.  src may be NULL.
 * Synchronises; returns KX_ERR_NONFINITE if f left the finite range.  On return with a mass
 * schedule, the handle's tensor is the one of the last stage evaluated. */
kx_status_t kx_evolve(kx_handle_t h, double* f, int32_t B, const kx_source_t* src,
                      const kx_evolve_t* ctl, void* stream);

/* Monoenergetic source (eq. 3.7): deposition of delta(p - p0) on the grid for the handle's current mass
 * (PAPER.md:171).  With p_L <= p0 <= p_R the neighbouring grid points and the energy-linear fractions
 * alpha_R = (E_0 - E_L)/(E_R - E_L), alpha_L = 1 - alpha_R, the shape G_L = alpha_L / h_L, G_R = alpha_R / h_R (0 elsewhere)
 * has sum_i h_i G_i = 1 and sum_i h_i E_i G_i = E_0 exactly: used as a row of kx_source_t.G with amp = (2 pi^2/g_chi) x
 * (injected number per unit tau), it reproduces the injected number and energy rates of eq. B.2 exactly.
 * G: DEVICE [N].  KX_ERR_INVALID_ARG unless p[0] <= p0 <= p[N-1].  Asynchronous. */
kx_status_t kx_delta_source(kx_handle_t h, double p0, double* G, void* stream);

/* The time integration of Sec. 4.2 in u = ln a (settings of PAPER.md:474):
 *     df/du = kappa_b R(u) C[f; m(u)] + sum_s amp_s G_s,   R(u) = rate0 exp(rate_slope (u - u0))        (eq. 4.9)
 *     m(u) = m exp(mass_slope (u - u0)), m = the handle's current mass: with comoving momenta q = a p the kinematics see the
 *     mass m a; mass_slope != 0 re-evaluates a1-a3 on the device at every stage (m(u) is computed on the
 *     device from the controller's u: a rejected step costs no host round trip).
 * Regime 1 (eps_switch > 0 and du_fixed > 0): "the self-scattering rate is negligible ... we set the self-collisions to zero
 * and evolve the distribution with a fourth-order Runge-Kutta method on fixed intervals in u" (steps of du_fixed; with source
 * rates constant in u the RK4 update is f + du sum_s amp_s G_s).  At u0 and after every fixed step the monitor
 *     Gamma_2->2 / H = kappa_b R(u) sum_i h_i loss_i[f; m(u)] / sum_i h_i f_i          (reading D16)
 * is evaluated on the device (one operator evaluation); at the first such point where the LARGEST member ratio exceeds
 * eps_switch (1e-2) the whole batch enters regime 2 there.  eps_switch <= 0: regime 2 from u0.
 * Regime 2: adaptive Heun.
 * Every attempted step is an Euler predictor f_P = f + du k1 and the Heun corrector f_H = f + du (k1 + k2)/2 (two
 * operator evaluations); err = max_{b,i} |f_H - f_P| / (atol + rtol max(|f|, |f_H|)) over the whole batch; the step is
 * accepted iff err <= 1, and du <- du clamp(safety / sqrt(err), 0.2, 5), du <= u1 - u (reading D15).
 * Error norm, accept/reject and the step-size update run on the device; the host only enqueues attempts (in chunks of
 * 8, reading the controller state between chunks) until u reaches u1 or max_steps attempts were made. */
typedef struct {
    double u0, u1;         /* integration interval, u1 > u0 */
    double du0;            /* first step (1e-4) */
    double rtol, atol;     /* 1e-2 and 2e-8 */
    double safety;         /* 0.9 */
    double rate0, rate_slope;
    const double* kappa;   /* HOST [B] per-member coupling multiplier; NULL => 1 */
    const double* amp;     /* HOST [src->nsrc] constant source rates per unit u (src->amp is not used); NULL => no sources */
    int32_t max_steps;     /* attempted Heun steps at most (> 0) */
    uint32_t flags;        /* KX_PROJECT */
    double mass_slope;     /* m(u) = m exp(mass_slope (u - u0)); 0 = static mass */
    double du_fixed;       /* regime 1: fixed interval in u (> 0 to enable regime 1) */
    double eps_switch;     /* regime 1 ends when Gamma_2->2/H exceeds this (1e-2); <= 0: no regime 1 */
} kx_adaptive_t;

typedef struct {
    double u, du;          /* where the integration stopped, the step it would take next */
    int64_t accepted, rejected;
    int32_t done;          /* 1 iff u reached u1 */
    int32_t switched;      /* 1 iff regime 2 was entered */
    double u_switch;       /* where (u1 if never) */
    int64_t fixed_steps;   /* regime-1 steps taken */
    double ratio;          /* Gamma_2->2/H of the last monitor point (largest member) */
} kx_adaptive_result_t;

/* f: DEVICE [B,N] in/out; src: only nsrc and G are read (may be NULL); result: HOST (may be NULL).  Synchronises.
 * KX_ERR_NONFINITE if f left the finite range.  With mass_slope != 0 the handle is left with the kinematics and the tensor
 * of m(u) at the u where the integration stopped (as after kx_set_mass). */
kx_status_t kx_evolve_adaptive(kx_handle_t h, double* f, int32_t B, const kx_source_t* src,
                               const kx_adaptive_t* ctl, kx_adaptive_result_t* result, void* stream);

/* Number of stored (i, n<=m) entries, bytes of tensor data one kx_collide streams (the tiled operand when
 * it is in use, else 20 bytes per entry), grid size.
 * Synchronises the device.  Any output pointer may be NULL. */
kx_status_t kx_info(kx_handle_t h, int64_t* nnz, int64_t* tensor_bytes, int32_t* n);

/* Copy the stored tensor to HOST arrays (testing the builder entry by entry): rowptr[N+1]; for entry e of
 * row i: W[e] = W_inm + W_imn (n<m) or W_inn; omega[e] = omega_R; nmj[e] = n | m<<10 | j_L<<20.
 * cap = capacity of W/omega/nmj in entries; fails with KX_ERR_INVALID_ARG if cap < nnz. */
kx_status_t kx_tensor_export(kx_handle_t h, int64_t cap, int64_t* rowptr, double* W, double* omega, uint32_t* nmj);

/* Copy the device kinematics to HOST arrays of length N (any may be NULL): E_i, K_i, h_i. */
kx_status_t kx_kinematics_export(kx_handle_t h, double* E, double* K, double* hw);

/* Allocate the workspaces, the task table and (KX_STORE_TILED) the launch plan for batches of up to B members now, so
 * that later kx_collide* calls with B' <= B only enqueue work (no cudaMalloc, no synchronisation). */
kx_status_t kx_reserve(kx_handle_t h, int32_t B, void* stream);

/* KX_STORE_TILED + LOG: number of (member, evaluation) pairs that took the exact fallback (their Chebyshev error bound
 * was not negligible, or f held an Inf/NaN) since the last call; resets the counter.  Synchronises the device. */
kx_status_t kx_fallback_members(kx_handle_t h, int64_t* count);

/* Measurement aid (bench.py): while enabled, every launch of the evaluation kernel (a4-a8, the dominant kernel)
 * is bracketed by two CUDA events recorded on the caller's stream.  kx_profile_read synchronises the device,
 * returns the summed kernel time in milliseconds and the number of launches since the last read, and resets. */
kx_status_t kx_profile(kx_handle_t h, int32_t enable);
kx_status_t kx_profile_read(kx_handle_t h, double* contract_ms, int64_t* launches);

/* Measurement aid (bench.py): while enabled, the evaluation kernel writes %globaltimer stamps (ns) of its phases, one
 * row of 32 slots per CTA (160 rows): 0 entry, 1 prologue done, 2 partials written, 3 grid barrier passed, 4 exact
 * fallback done, 5 finishing phase done, 8..15 end of each gain warp's stream (tensor-core path).  kx_trace_read copies
 * the stamps of the launches since the last read (later launches overwrite earlier ones) to HOST stamps[160*32],
 * zero = not written, and clears them.  Synchronises the device. */
kx_status_t kx_trace(kx_handle_t h, int32_t enable);
kx_status_t kx_trace_read(kx_handle_t h, uint64_t* stamps);

/* Measurement aid (bench.py): peak FP64 throughput of `device` in TFLOP/s, register-resident chains without memory
 * traffic.  kind 0 = DFMA (plain FP64 pipe), 1 = DMMA.8x8x4 (FP64 tensor pipe, the instruction of the tiled
 * contraction).  Synchronises the device; takes about 50 ms. */
kx_status_t kx_probe_flops(int device, int32_t kind, double* tflops);

/* Test aid, HOST only (no device is touched): the launch plan of the tensor-core kernel for a grid of N points, a batch of
 * B members, Q loss nodes per bracket and `sm_count` SMs, given the number of gain groups of every 16-row tile
 * (groups_per_tile[ceil(N/16)]).  head[8] = {gain CTAs, loss CTAs, member tiles per pass, loss window in chunks, tiles,
 * supertiles, loss chunks, dynamic shared memory in bytes}; wstart[tiles + 1] = first gain warp of every tile (8 warps per
 * CTA); ld[8] = first / last loss CTA of each of the (up to 4) supertiles.  tests/test_plan_cpu.py checks the invariants the
 * kernel relies on (every gain warp owns at least one group, every partial slot that is summed was written, every CTA fits). */
kx_status_t kx_plan_probe(int32_t N, int32_t B, int32_t Q, int32_t sm_count, const uint32_t* groups_per_tile,
                          int32_t* head, uint32_t* wstart, uint32_t* ld);

const char* kx_last_error(kx_handle_t h);   /* h may be NULL: returns the last build failure */
void        kx_destroy(kx_handle_t h);
int32_t     kx_version(void);

#ifdef __cplusplus
}
#endif
#endif /* KX_H_ */
