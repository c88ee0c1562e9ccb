// kx_internal.cuh -- shared declarations of libkx's translation units (NOT part of the ABI).
// The CUDA path shares nothing with oracle/: no header, table, constant generator or helper.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string>
#include <utility>
#include <vector>

#include "../../include/kx.h"

#define KX_MAX_N      1024     // n, m, j_L are packed 10 bits each
#define KX_MAX_SRC    8
#define KX_CTA        256      // threads per CTA of the contraction kernels
#define KX_EXP_BITS   8        // 2^8-entry exp2 table
#define KX_EXP_REP    16       // table replicated once per bank pair: conflict-free 64-bit gathers
#define KX_TI         16       // rows i per tile of the tiled (DMMA) storage: two 8-row MMA blocks
#define KX_QMAX       32       // largest number of Chebyshev nodes of the compressed LOG loss term
#define KX_GROUP_DBL  256      // doubles of tensor data per group: 4 quads x 2 row blocks x 32 lanes
#define KX_TRACE_CTAS  160      // clock-stamp trace (kx_trace): CTAs x slots of 8 bytes
#define KX_TRACE_SLOTS 32
#define KX_FB_BT      4        // members per group of the exact fallback inside the DMMA kernel
#define KX_BLUT_MAX   4096     // entries of the bracket look-up table (64 keys per binade of K)

// Device-side view of a handle: plain pointers, passed by value to every kernel.
struct KxDev {
    int N;
    int interp;          // KX_INTERP_*
    int exp_impl;        // KX_EXP_*
    int eta;             // KX_STAT_*: 0, +1 (Bose), -1 (Fermi)
    int prec;            // KX_FP64 | KX_FP32 (arithmetic of the streaming contraction)
    int n_mu;            // > 0: numerical angular kernel with n_mu Gauss-Legendre nodes (gl_mu, gl_w)
    const double *gl_mu, *gl_w;
    int chunk;           // entries per contraction task
    double m, g_chi, M2_0, m_med, f_floor, eps_supp;
    const double* m_dev;      // not null: the kinematic mass is read from the device (kx_evolve_adaptive with m(u)); else `m`
    // grid and kinematics [N]
    const double *p, *dp;
    double *E, *K, *h;        // eq. B.1; K_i = E_i - m evaluated as p^2/(E+m)
    double *invdK;            // 1/(K_{j+1}-K_j), j < N-1
    double *arow;             // 1/(2 E_i g_chi) * 1/(64 pi^3 p_i)
    double *ccol;             // dp_n p_n / E_n
    // run table of the builder [N*N]: for (i,n) the valid m form one interval [mlo, mlo+len)
    int *run_mlo, *run_len;
    unsigned *run_off;        // [N*N+1] exclusive scan of run_len; run_off[N*N] = nnz
    // row-compressed symmetric tensor
    unsigned *rowptr;         // [N+1]
    double *W;                // [cap] W_inm + W_imn (n<m) or W_inn
    double *omega;            // [cap] omega_R of eq. B.19
    unsigned *nmj;            // [cap] n | m<<10 | jL<<20
    // contraction tasks: row i is cut into ceil(len_i/chunk) tasks
    unsigned *taskptr;        // [N+1] exclusive scan; taskptr[N] = ntasks
    const double *exptab;     // [2^KX_EXP_BITS] 2^(k/2^KX_EXP_BITS)
    unsigned *blut;           // bracket look-up table of k_fill (kx_build.cu): [0] first key, [1] size, [2..] lower bound of j_L per key
};

// Tiled storage (KX_STORE_TILED), the operands of the DMMA contraction kernel (kx_tiled.cu).
//
// Both terms have the form  out[b, i] += sum_k X[b, k] * A[k, i]  (k in quads of 4 = one DMMA.8x8x4).
//
//   gain:  rows i are cut into tiles of KX_TI = 16.  k = (n, m) with n <= m;  A = W_inm + W_imn (0 where the triple
//          is dropped for row i), X = f_n f_m.  For fixed (tile, n) the m with any kept row form one interval: a
//          "run", padded to a multiple of 4.  A group (4 quads) stores its 256 doubles in MMA-fragment order
//          [quad][row block rb][lane], the lane's element being A[k = 4 quad + lane%4][i = 16 t + 8 rb + lane/4].
//          desc[quad] = m0 | n << 20: the rows of f^T holding f_m for the quad (m0..m0+3) and the row that scales
//          them (f_n; padding quads: 0 | N << 20, the column of ones, with A = 0).  vtptr[t] = first group of tile t.
//   loss:  k = (j, c), c < Q;  A = M_c(i,j) = sum_{(n<=m) in bracket j of row i} Wsym T_c(2 omega_R - 1)
//          (Chebyshev moments of the bucket), X = a_c(b,j) = Chebyshev coefficients of the degree-(Q-1) interpolant
//          of omega -> f_j^(1-omega) f_(j+1)^omega (LOG) or the exact two coefficients (LINEAR, Q = 2).  The operand
//          is dense: AL[chunk kc][8-row block][quad][lane] holds A[k = 16 kc + 4 quad + lane%4][i = 8 block + lane/4],
//          so that a chunk of 16 k for 256 consecutive rows (a "supertile") is one contiguous 32 KiB piece.
struct KxTiled {
    int NT;                   // number of gain tiles = ceil(N / 16)
    int Q;                    // Chebyshev coefficients per bracket (LINEAR: 2)
    int LC;                   // loss chunks of 16 k = ceil((N-1) Q / 16)
    int NR8;                  // 8-row blocks = ceil(N / 8)
    int RS;                   // 256-row supertiles = ceil(N / 256)
    int *trun_mlo;            // [NT*N] first m of the run (tile, n)
    unsigned *trun_q;         // [NT*N] quads of the run
    unsigned *trun_off;       // [NT*(N+1)] exclusive scan of trun_q inside the tile; [t*(N+1)+N] = quads of tile t
    unsigned *vtptr;          // [NT + 1] exclusive scan of gain groups per tile
    double *A;                // [groups][256]   gain operand
    unsigned *desc;           // [groups][4]
    double *AL;               // [LC][NR8][128]  loss operand
    const double *dct;        // [Q*Q] (2 - delta_c0)/Q cos(c theta_q), theta_q = (2q+1) pi / (2Q)
    const double *nodes;      // [Q] omega_q = (1 + cos theta_q)/2
    double flag_log2;         // log2(2 / Q!) ... see the loss role of k_dmma (kx_tiled.cu)
};

// Plan of one launch of the DMMA kernel (made on the host by kx_dmma_plan, passed by value).
//   CTAs [0, GG) take the gain role, [GG, GG + GL) the loss role.  Gain warp w (global index = CTA * 8 + warp) works on
//   ONE tile: the warps [wstart[t], wstart[t+1]) share the groups of tile t in equal contiguous ranges (a warp never
//   crosses a tile, so a CTA adds the accumulators of its warps in shared memory and writes one partial per tile it
//   touches, slot = CTA + tile).  Warps beyond wstart[NT] are idle.
#define KX_MAX_NT 64
struct KxPlan {
    int nbt;                  // member tiles (of 8) per pass
    int GG, GL;               // CTAs per role
    int WC;                   // chunks of 16 k whose Chebyshev coefficients a loss CTA holds at a time
    unsigned wstart[KX_MAX_NT + 1];
    unsigned vt[KX_MAX_NT + 1];      // copy of vtptr: first group of every tile
    unsigned ld0[4], ld1[4];         // first / last loss CTA (relative to GG) that worked on supertile sp (RS <= 4)
};

struct KxAdapt;
struct kx_handle_s {
    KxDev d;
    int device;
    int sm_count;
    long long cap;            // capacity of W/omega/nmj in entries
    long long nnz;            // host copy, valid when !nnz_stale
    KxTiled t;                // tiled storage (valid when tiled_ok)
    int storage;              // KX_STORE_*
    bool tiled_ok;            // t.A / t.desc describe the current kinematics
    long long cap_groups;     // capacity of t.A / t.desc in groups
    long long groups;         // host copy of vtptr[NT]
    int ws_xstride;           // members per partial slot (batch capacity padded)
    long long *mstat;         // [2][wsB][2] per member, double-buffered by launch parity: ordered key of the largest
                              // interpolation-error term over the brackets, bits of max_i |f_i| (see kx_member_flagged)
    double *gpart;            // [ws_xstride, sm_count + NT + 1, 16]  gain partials of the DMMA kernel (one per CTA and tile), member-major:
    double *lpart;            // [ws_xstride, sm_count + RS + 1, 256] loss partials (one per CTA and supertile); a member's slots are contiguous
    std::vector<unsigned> vt_host;   // host copy of vtptr [NT + 1] (the plan of the DMMA kernel is made on the host)
    KxPlan plan;              // role split and warp -> tile map of the DMMA kernel for batch plan_B
    int plan_B;               // 0 = no plan
    unsigned *bar;            // device [4]: grid barrier of the fused kernels (arrival count, released epoch), fallback count
    unsigned epoch;           // launch serial number of the fused kernels (two barrier epochs per launch)
    unsigned bar_total;       // CTAs that have arrived at bar[3] once every launch enqueued so far has run
    unsigned long long *trace;       // device [KX_TRACE_CTAS][KX_TRACE_SLOTS] clock stamps of the last fused launch, or null
    bool tracing;
    void *tiled_blob;         // one allocation holding the small tables of KxTiled
    bool nnz_stale;
    int chunk_for_B;          // the batch size taskptr was last built for (0 = none)
    // workspaces, grown on demand
    int wsB;                  // batch capacity of the buffers below
    long long ws_tasks;       // task capacity of `part`
    double *yd;               // [wsB, N, 2]  LOG: (log2 f_j, log2 f_{j+1} - log2 f_j); LINEAR: (f_j, f_{j+1}-f_j)
    double *part;             // [ws_tasks, wsB, 2] per-task partial (gain, loss frequency)
    double *fstage, *k1, *k2, *k3, *Cbuf;   // [wsB, N] evolve buffers
    double *hostio;           // [wsB, N] x2 staging for kx_collide_host
    double *runbuf;           // device copy of tau / rate / amp of a one-launch kx_evolve (grown on demand)
    size_t runbuf_cap;        // in doubles
    int *flag;                // device non-finite flag
    KxAdapt *adapt;           // device controller state of kx_evolve_adaptive
    double p_lo, p_hi;        // host copies of p[0], p[N-1]
    double *gl;               // device [2 n_mu]: Gauss-Legendre nodes and weights (n_mu > 0)
    void *dev_blob;           // one allocation holding the [N]-sized arrays
    bool profiling;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> prof_events;
    size_t prof_used;
    std::string err;
};

#define KX_CUDA(call)                                                                          \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess) {                                                               \
            char buf_[512];                                                                    \
            snprintf(buf_, sizeof buf_, "%s:%d: %s -> %s", __FILE__, __LINE__, #call,           \
                     cudaGetErrorString(e_));                                                  \
            h->err = buf_;                                                                     \
            return KX_ERR_CUDA;                                                                \
        }                                                                                      \
    } while (0)

// ---- cooperative launch: every CTA of the grid is resident at the same time, so the grid barrier of the fused
// kernels (kx_device.cuh) cannot deadlock.  The launch fails (cudaErrorCooperativeLaunchTooLarge) instead of hanging
// if the grid does not fit.
template <typename... KArgs, typename... Args>
inline cudaError_t kx_launch_coop(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s,
                                  Args&&... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeCooperative;
    at[0].val.cooperative = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}
#ifdef __CUDACC__

// ---------------------------------------------------------------- exp2 for the LOG loss term
// 2^t = 2^k * T[idx] * 2^r,  t = k + idx/256 + r, |r| <= 2^-9.  Adding 1.5*2^44 leaves round(256 t) in the
// low mantissa bits (one DADD), T is a 256-entry table in shared memory (entry k at tab[k * STRIDE]; the streaming
// kernel replicates it 16x so that its 64-bit gathers are bank-conflict free), 2^r = 1 + r q(r) with q the degree-3 Chebyshev interpolant of
// (2^r-1)/r on |r| <= 1.01*2^-9 (polynomial error 5e-18), and 2^k is added to the exponent field by the
// integer pipe.  FP64-pipe cost: 2 DADD + 1 DADD + 3 DFMA + 1 DMUL + 1 DFMA = 8.  Valid for
// -1021 < t < 1023 (f_floor >= 1e-300 keeps t >= -997).
template <int STRIDE>
__device__ __forceinline__ double kx_exp2_tab(double t, const double* __restrict__ tab_lane)
{
    const double MAG = 26388279066624.0;                 // 1.5 * 2^44
    const double C1 = 0.6931471805599427, C2 = 0.24022650695910042,
                 C3 = 0.05550411385340617, C4 = 0.009618129707037269;
    double tm = t + MAG;
    int nlo = __double2loint(tm);
    double r = t - (tm - MAG);
    double T = tab_lane[(nlo & ((1 << KX_EXP_BITS) - 1)) * STRIDE];
    double q = fma(fma(fma(C4, r, C3), r, C2), r, C1);
    double s = r * q;
    double res = fma(T, s, T);
    int hi = __double2hiint(res) + ((nlo >> KX_EXP_BITS) << 20);
    return __hiloint2double(hi, __double2loint(res));
}


// Per-member statistics of the tiled LOG path, accumulated with atomicMax by the loss role of k_dmma (order independent, so the
// result is deterministic):  mstat[2b] = key(max over brackets j of  log2 max(f_j, f_j+1) + Q (log2 |ln(f_j+1/f_j)| - 2)
// + log2(2/Q!)),  mstat[2b+1] = bits of max_i |f_i|.  key() maps doubles to integers of the same order.
#define KX_MSTAT_NONE (-0x7fffffffffffffffLL - 1)
__device__ __forceinline__ long long kx_dkey(double x)
{
    const long long b = __double_as_longlong(x);
    return b >= 0 ? b : (b ^ 0x7fffffffffffffffLL);
}
// A member takes the exact streaming path when the interpolation error bound of some bracket,
//     2 (|ln(f_(j+1)/f_j)|/4)^Q / Q! * max(f_j, f_(j+1)),   exceeds 1e-15 max_i f_i      (kxd::member_flagged, kx_device.cuh)
#endif

// ---- launchers implemented in kx_build.cu
cudaError_t kx_launch_kinematics(const KxDev& d, double m, cudaStream_t s);
cudaError_t kx_launch_runs(const KxDev& d, cudaStream_t s);      // run table + scan + rowptr
cudaError_t kx_launch_fill(const KxDev& d, cudaStream_t s);      // W, omega, nmj
cudaError_t kx_launch_tasks(const KxDev& d, int chunk, cudaStream_t s);

// ---- launchers implemented in kx_contract.cu
// controller state of kx_evolve_adaptive, on the device
struct KxAdapt {
    double u, du;
    long long errkey;        // ordered key (kx_dkey) of the largest scaled error of the attempt, atomicMax over the CTAs
    long long accepted, rejected;
    int done;
    // regime 1 of Sec. 4.2 (sources only on fixed intervals, Gamma_2->2/H monitored)
    int switched;            // the largest member ratio exceeded eps_switch at u_switch
    long long fixed_steps;
    double u_switch, ratio;  // ratio: Gamma_2->2/H of the last monitor point (largest member)
};

struct KxStage {             // what the finishing kernel does after the reduction
    unsigned flags;          // KX_PROJECT
    double *C, *gain, *loss, *diag;       // outputs of kx_collide_ex (any may be null); diag stride 4
    int diag_stride;
    // evolve: mode 0 = none; otherwise the Runge-Kutta update below
    int rk_method, rk_stage;
    double dt, rate;
    const double *kappa;     // device [B] or null
    int nsrc;
    const double *G;         // device [nsrc,N]
    double amp[KX_MAX_SRC];
    double *f;               // state [B,N]
    double *fstage;          // stage input written by this stage for the next one
    double *k1, *k2, *k3;
    double *ydnext;          // where to write yd of the next stage input (fused prep) or null
    // tiled path: partials of the DMMA phase; flagged members (kx_member_flagged) take the streaming partials instead
    double *gpart;           // [slots, xstride, 16] or null (streaming path only)
    double *lpart;           // [slots, xstride, 256]
    long long *mstat;        // this launch's member statistics [B][2], or null (LINEAR: no fallback)
    long long *mstat_next;   // the other buffer: reset (all mstat_cap members) by the finishing phase for the next launch
    int mstat_cap;
    int NT, LC, RS, xstride;
    int gslots, lslots;      // partial slots per member: gpart [member][gslots][16], lpart [member][lslots][256]
    int *flag;
    int evolve;
    double *part;            // [tasks, B, 2 or 4] partials of the exact streaming contraction
    // grid barrier of the fused kernels (kx_device.cuh) and the optional clock-stamp trace
    unsigned *bar;           // [0] arrivals, [1] released epoch (second barrier of a launch); [2] fallback count; [3] growing counter
    unsigned epoch;
    unsigned bar_target;     // value of bar[3] when every CTA of this launch has arrived at the first barrier
    unsigned long long *trace;
    unsigned *fb_count;      // device counter: members evaluated by the exact fallback (kx_fallback_count)
    // adaptive Heun (rk_method == KX_HEUN_ADAPT): dt and the rate come from the device controller state
    KxAdapt *ad;
    double ad_u0, ad_rate0, ad_slope, ad_rtol, ad_atol;
};
#define KX_HEUN_ADAPT 3      // internal: Euler predictor / Heun corrector with the error norm of kx_evolve_adaptive
// one operator evaluation on the exact streaming path: y = log2 f, contraction, grid barrier, finishing phase: ONE kernel
// (bar_total: the handle's running count of barrier arrivals; the launcher adds its grid size and sets st.bar_target)
cudaError_t kx_launch_stream(const KxDev& d, int sm_count, const double* f, const double* yd, int B,
                             KxStage st, unsigned* bar_total, cudaStream_t s);
// a whole fixed-step integration (static mass, no diagnostics) on the exact streaming path in ONE cooperative launch
// step data of a one-launch integration (k_stream_run), on the device
struct KxRun {
    int method, S;            // KX_EULER | KX_HEUN | KX_RK4, number of steps
    const double* tau;        // device [S+1]
    const double* rate;       // device [2S+1] or null
    const double* amp;        // device [nsrc, S] or null
};
// the streaming kernels are instantiated per member-group size BT in kx_stream_bt{1,2,4,8}.cu (compiled in parallel)
cudaError_t kx_launch_stream_bt1(const KxDev& d, int sm_count, const double* f, const double* yd, int B, KxStage& st, unsigned* bar_total, cudaStream_t s, const KxRun* run);
cudaError_t kx_launch_stream_bt2(const KxDev& d, int sm_count, const double* f, const double* yd, int B, KxStage& st, unsigned* bar_total, cudaStream_t s, const KxRun* run);
cudaError_t kx_launch_stream_bt4(const KxDev& d, int sm_count, const double* f, const double* yd, int B, KxStage& st, unsigned* bar_total, cudaStream_t s, const KxRun* run);
cudaError_t kx_launch_stream_bt8(const KxDev& d, int sm_count, const double* f, const double* yd, int B, KxStage& st, unsigned* bar_total, cudaStream_t s, const KxRun* run);
bool kx_stream_run_supported(const KxDev& d);      // built for the default fp64 paths only (LOG table exp2, LINEAR; classical)
cudaError_t kx_launch_stream_run(const KxDev& d, int sm_count, double* f, int B, KxStage st, int method, int S,
                                 const double* tau_dev, const double* rate_dev, const double* amp_dev,
                                 unsigned* bar_total, cudaStream_t s);
cudaError_t kx_launch_adapt_step(const KxDev& d, double* f, const double* fnew, int B, KxAdapt* ad, double u1, double safety,
                                 int* flag, cudaStream_t s);      // accept/reject + controller update
cudaError_t kx_launch_delta_source(const KxDev& d, double p0, double* G, cudaStream_t s);
// m(u) of the adaptive integrator on the device: *m_dev = mass0 exp(slope (u_stage - u0)), u_stage = ad->u (+ ad->du)
cudaError_t kx_launch_adapt_mass(KxAdapt* ad, int stage, double u0, double mass0, double slope, double* m_dev, cudaStream_t s);
// regime 1: monitor Gamma_2->2/H at ad->u (switch / stop), then one sources-only step of at most du_fixed
cudaError_t kx_launch_regime1_step(const KxDev& d, double* f, const double* loss, int B, const double* kappa, int nsrc,
                                   const double* G, const double* amp_dev, KxAdapt* ad, double u0, double u1, double du_fixed,
                                   double eps_switch, double rate0, double rate_slope, cudaStream_t s);
cudaError_t kx_launch_moments(const KxDev& d, const double* f, int B, double* n, double* rho,
                              double* p1, double* p2, int stride, cudaStream_t s);
// ---- tiled path (kx_tiled_build.cu, kx_tiled.cu)
cudaError_t kx_launch_tile_runs(const KxDev& d, const KxTiled& t, cudaStream_t s);     // runs, scans, vtptr
cudaError_t kx_launch_tile_fill(const KxDev& d, const KxTiled& t, cudaStream_t s);     // A, desc (gain + loss)
// one operator evaluation on the tensor-core path: DMMA phase, grid barrier, (exact fallback, barrier,) finishing phase
cudaError_t kx_launch_dmma(const KxDev& d, const KxTiled& t, const KxPlan& plan, const double* f, int B,
                           KxStage st, unsigned* bar_total, cudaStream_t s);
cudaError_t kx_dmma_configure(); // shared-memory attributes of every instantiation (once per process)
int kx_xstride(int B);
void kx_dmma_plan(const KxDev& d, const KxTiled& t, int sm_count, const unsigned* vt_host, int B, KxPlan* plan);
int kx_pick_bt(int N, int B);
int kx_pick_chunk(long long nnz_est, int N, int B, int sm_count);
