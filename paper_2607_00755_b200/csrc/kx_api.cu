// kx_api.cu -- the C ABI of include/kx.h: argument checks, memory ownership and launch sequencing.
// All arithmetic of the path runs in the kernels of kx_build.cu / kx_contract.cu; nothing here computes
// a physical quantity on the host except the 256-entry exp2 table (a constant, not data dependent).
#include "kx_internal.cuh"

#include <math.h>
#include <stdlib.h>
#include <new>
#include <vector>

namespace {

thread_local std::string g_build_err;     // last kx_build failure of the calling thread (there is no handle yet)

struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
        if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

inline long long tri_entries(int N) { return (long long)N * ((long long)N * (N + 1) / 2); }

template <typename T>
cudaError_t dalloc(T** p, size_t count) { return cudaMalloc((void**)p, count * sizeof(T)); }

void free_tensor(kx_handle_s* h)
{
    cudaFree(h->d.W); cudaFree(h->d.omega); cudaFree(h->d.nmj);
    h->d.W = nullptr; h->d.omega = nullptr; h->d.nmj = nullptr;
    h->cap = 0;
}

kx_status_t alloc_tensor(kx_handle_s* h, long long cap)
{
    free_tensor(h);
    if (cap < 1) cap = 1;
    KX_CUDA(dalloc(&h->d.W, (size_t)cap));
    KX_CUDA(dalloc(&h->d.omega, (size_t)cap));
    KX_CUDA(dalloc(&h->d.nmj, (size_t)cap));
    h->cap = cap;
    return KX_OK;
}

void free_tiled(kx_handle_s* h)
{
    cudaFree(h->t.A); cudaFree(h->t.desc);
    h->t.A = nullptr; h->t.desc = nullptr;     // t.AL has a fixed size: freed in kx_destroy
    h->cap_groups = 0; h->tiled_ok = false;
}

kx_status_t alloc_tiled(kx_handle_s* h, long long groups)
{
    free_tiled(h);
    if (groups < 1) groups = 1;
    KX_CUDA(dalloc(&h->t.A, (size_t)groups * KX_GROUP_DBL));
    KX_CUDA(dalloc(&h->t.desc, (size_t)groups * 4));
    h->cap_groups = groups;
    return KX_OK;
}

// a2-a3 in the tiled layout for the current kinematics (the run table of kx_launch_runs must be current).
// Synchronises the stream (the group count decides the allocation) and may reallocate the gain operand.
kx_status_t build_tiled(kx_handle_s* h, cudaStream_t s)
{
    KX_CUDA(kx_launch_tile_runs(h->d, h->t, s));
    h->vt_host.assign((size_t)h->t.NT + 1, 0u);
    KX_CUDA(cudaMemcpyAsync(h->vt_host.data(), h->t.vtptr, ((size_t)h->t.NT + 1) * 4, cudaMemcpyDeviceToHost, s));
    KX_CUDA(cudaStreamSynchronize(s));
    const unsigned g = h->vt_host[h->t.NT];
    h->groups = g;
    if (h->cap_groups < (long long)g) {
        kx_status_t rc = alloc_tiled(h, g);
        if (rc != KX_OK) return rc;
    }
    KX_CUDA(cudaMemsetAsync(h->t.A, 0, (size_t)h->groups * KX_GROUP_DBL * 8, s));
    KX_CUDA(kx_launch_tile_fill(h->d, h->t, s));
    h->tiled_ok = true;
    h->plan_B = 0;
    return KX_OK;
}

void free_ws(kx_handle_s* h)
{
    cudaFree(h->yd); cudaFree(h->part); cudaFree(h->fstage); cudaFree(h->k1); cudaFree(h->k2);
    cudaFree(h->k3); cudaFree(h->Cbuf); cudaFree(h->hostio);
    cudaFree(h->mstat); cudaFree(h->gpart); cudaFree(h->lpart);
    h->yd = h->part = h->fstage = h->k1 = h->k2 = h->k3 = h->Cbuf = h->hostio = nullptr;
    h->gpart = h->lpart = nullptr; h->mstat = nullptr;
    h->wsB = 0; h->ws_tasks = 0; h->ws_xstride = 0;
}

// the smallest chunk is 1024 entries, so a row of len entries has at most len/1024+1 tasks
inline long long max_tasks(const kx_handle_s* h) { return h->cap / 1024 + h->d.N + 1; }

kx_status_t ensure_ws(kx_handle_s* h, int B)
{
    const long long need_tasks = max_tasks(h);
    if (B <= h->wsB && need_tasks <= h->ws_tasks) return KX_OK;
    const int nB = B > h->wsB ? B : h->wsB;
    free_ws(h);
    const size_t bn = (size_t)nB * h->d.N;
    KX_CUDA(dalloc(&h->yd, bn * 2));
    KX_CUDA(dalloc(&h->part, (size_t)need_tasks * nB * 4));      // 2 sums per (task, member); 4 with quantum statistics
    KX_CUDA(dalloc(&h->fstage, bn));
    KX_CUDA(dalloc(&h->k1, bn));
    KX_CUDA(dalloc(&h->k2, bn));
    KX_CUDA(dalloc(&h->k3, bn));
    KX_CUDA(dalloc(&h->Cbuf, bn + (size_t)nB));   // + kappa[B]
    KX_CUDA(dalloc(&h->hostio, bn * 2));
    if (h->storage == KX_STORE_TILED) {
        const int xs = kx_xstride(nB);
        KX_CUDA(dalloc(&h->mstat, (size_t)nB * 4));           // two buffers, used alternately (launch parity)
        {
            std::vector<long long> init((size_t)nB * 4);
            for (int b = 0; b < 2 * nB; ++b) { init[2 * b] = (-0x7fffffffffffffffLL - 1); init[2 * b + 1] = 0; }
            KX_CUDA(cudaMemcpy(h->mstat, init.data(), init.size() * 8, cudaMemcpyHostToDevice));
        }
        KX_CUDA(dalloc(&h->gpart, (size_t)(h->sm_count + h->t.NT + 1) * xs * 16));
        KX_CUDA(dalloc(&h->lpart, (size_t)(h->sm_count + h->t.RS + 1) * xs * 256));
        h->ws_xstride = xs;
        h->plan_B = 0;
    }
    h->wsB = nB; h->ws_tasks = need_tasks;
    // test aid (tests/test_gpu_parity.py): KX_POISON_WS=1 fills every partial-sum workspace with NaN bit patterns, so that a
    // slot the kernels read without having written it shows up in the result instead of passing on freshly zeroed memory
    if (const char* e = getenv("KX_POISON_WS"); e && e[0] == '1') {
        KX_CUDA(cudaMemset(h->part, 0xFF, (size_t)need_tasks * nB * 4 * 8));
        KX_CUDA(cudaMemset(h->yd, 0xFF, bn * 2 * 8));
        if (h->gpart) KX_CUDA(cudaMemset(h->gpart, 0xFF, (size_t)(h->sm_count + h->t.NT + 1) * h->ws_xstride * 16 * 8));
        if (h->lpart) KX_CUDA(cudaMemset(h->lpart, 0xFF, (size_t)(h->sm_count + h->t.RS + 1) * h->ws_xstride * 256 * 8));
    }
    return KX_OK;
}

// Integrators on small problems are bound by kernel launches, not by work: below this many (entry, member) pairs per
// operator evaluation the exact streaming path (2 kernels per stage) beats the tensor-core path (5 kernels per stage);
// measured: cfg1 12 vs 21 us per stage, cfg2 16 vs 23 us, N=256 B=4 76 vs 33 us.
constexpr long long kSmallProblem = 1500000;

long long nnz_estimate(const kx_handle_s* h)
{
    if (!h->nnz_stale) return h->nnz;
    return (long long)(0.66 * (double)tri_entries(h->d.N));
}

// (re)build the task table when the chunk size changes or the tensor was rebuilt
kx_status_t ensure_tasks(kx_handle_s* h, int B, cudaStream_t s)
{
    const int chunk = kx_pick_chunk(nnz_estimate(h), h->d.N, B, h->sm_count);
    if (chunk != h->d.chunk || h->chunk_for_B == 0) {
        h->d.chunk = chunk;
        KX_CUDA(kx_launch_tasks(h->d, chunk, s));
        h->chunk_for_B = B;
    }
    return KX_OK;
}

// a1-a3 for mass m; the capacity must already cover the result
kx_status_t rebuild(kx_handle_s* h, double m, cudaStream_t s)
{
    h->d.m = m;
    KX_CUDA(kx_launch_kinematics(h->d, m, s));
    KX_CUDA(kx_launch_runs(h->d, s));
    KX_CUDA(kx_launch_fill(h->d, s));
    h->nnz_stale = true;
    h->chunk_for_B = 0;
    h->tiled_ok = false;
    return KX_OK;
}

// the tiled operand is rebuilt lazily: kx_set_mass and mass schedules only refresh the streaming storage
kx_status_t ensure_tiled(kx_handle_s* h, cudaStream_t s)
{
    if (h->storage != KX_STORE_TILED || h->tiled_ok) return KX_OK;
    return build_tiled(h, s);
}

// One operator evaluation (a4-a8) = ONE cooperative kernel: the caller has filled the outputs and the Runge-Kutta fields
// of *st; this adds the path's buffers, the barrier epoch and the trace pointer and launches.
kx_status_t launch_step(kx_handle_s* h, const double* f, int B, bool have_yd, bool use_tiled, KxStage* st, cudaStream_t s)
{
    if (h->profiling) {
        if (h->prof_used == h->prof_events.size()) {
            cudaEvent_t a, b;
            KX_CUDA(cudaEventCreate(&a));
            KX_CUDA(cudaEventCreate(&b));
            h->prof_events.emplace_back(a, b);
        }
        KX_CUDA(cudaEventRecord(h->prof_events[h->prof_used].first, s));
    }
    st->part = h->part;
    st->bar = h->bar;
    st->fb_count = h->bar + 2;
    h->epoch += 2;                   // two barrier epochs per launch
    st->epoch = h->epoch;
    st->trace = h->tracing ? h->trace : nullptr;
    if (use_tiled) {
        if (h->plan_B != B) {
            kx_dmma_plan(h->d, h->t, h->sm_count, h->vt_host.data(), B, &h->plan);
            h->plan_B = B;
        }
        const int par = (int)((h->epoch >> 1) & 1u);
        st->gpart = h->gpart; st->lpart = h->lpart; st->xstride = h->ws_xstride;
        st->gslots = h->sm_count + h->t.NT + 1; st->lslots = h->sm_count + h->t.RS + 1;
        st->mstat = nullptr; st->mstat_next = nullptr; st->mstat_cap = 0;
        if (h->d.interp == KX_INTERP_LOG) {      // LINEAR is exact: no statistics, no fallback
            st->mstat = h->mstat + (size_t)par * h->wsB * 2;
            st->mstat_next = h->mstat + (size_t)(1 - par) * h->wsB * 2;
            st->mstat_cap = h->wsB;
        }
        st->NT = h->t.NT; st->LC = h->t.LC; st->RS = h->t.RS;
        KX_CUDA(kx_launch_dmma(h->d, h->t, h->plan, f, B, *st, &h->bar_total, s));
    } else {
        st->gpart = nullptr; st->lpart = nullptr; st->mstat = nullptr; st->mstat_next = nullptr;
        KX_CUDA(kx_launch_stream(h->d, h->sm_count, f, have_yd ? h->yd : nullptr, B, *st, &h->bar_total, s));
    }
    if (h->profiling) {
        KX_CUDA(cudaEventRecord(h->prof_events[h->prof_used].second, s));
        h->prof_used++;
    }
    return KX_OK;
}

kx_status_t check_batch(kx_handle_s* h, const void* f, int B)
{
    if (!f || B < 1) { h->err = "f is NULL or B < 1"; return KX_ERR_INVALID_ARG; }
    if (((uintptr_t)f & 15u) != 0) { h->err = "device pointer not 16-byte aligned"; return KX_ERR_INVALID_ARG; }
    return KX_OK;
}

kx_status_t collide_impl(kx_handle_s* h, const double* f, double* C, double* gain, double* loss, double* diag,
                         int B, unsigned flags, cudaStream_t s)
{
    kx_status_t rc = check_batch(h, f, B);
    if (rc != KX_OK) return rc;
    if (C == f) { h->err = "in-place kx_collide (C == f) is not allowed"; return KX_ERR_INVALID_ARG; }
    if ((rc = ensure_ws(h, B)) != KX_OK) return rc;
    if ((rc = ensure_tasks(h, B, s)) != KX_OK) return rc;
    if ((rc = ensure_tiled(h, s)) != KX_OK) return rc;
    KxStage st = {};
    st.flags = flags & KX_PROJECT;
    st.C = C; st.gain = gain; st.loss = loss; st.diag = diag; st.diag_stride = 4;
    st.evolve = 0;
    return launch_step(h, f, B, false, h->storage == KX_STORE_TILED, &st, s);
}

}  // namespace

extern "C" {

int32_t kx_version(void) { return 100; }

const char* kx_last_error(kx_handle_t h) { return h ? h->err.c_str() : g_build_err.c_str(); }

void kx_destroy(kx_handle_t h)
{
    if (!h) return;
    {
        DeviceGuard g(h->device);
        free_tensor(h);
        free_tiled(h);
        free_ws(h);
        cudaFree(h->dev_blob);
        cudaFree(h->tiled_blob);
        cudaFree(h->t.AL);
        cudaFree(h->adapt);
        cudaFree(h->bar);
        cudaFree(h->trace);
        cudaFree(h->gl);
        cudaFree(h->runbuf);
        for (auto& ev : h->prof_events) { cudaEventDestroy(ev.first); cudaEventDestroy(ev.second); }
    }
    delete h;
}

kx_status_t kx_build(const kx_grid_t* grid, const kx_species_t* sp, const kx_msq_t* msq,
                     const kx_opts_t* opts, int device, void* stream, kx_handle_t* out)
{
    if (out) *out = nullptr;
    if (!grid || !sp || !msq || !out || !grid->p || !grid->dp) { g_build_err = "null argument"; return KX_ERR_INVALID_ARG; }
    const int N = grid->n;
    if (N < 4) { g_build_err = "N must be at least 4"; return KX_ERR_INVALID_ARG; }
    if (N > KX_MAX_N) { g_build_err = "N > 1024 is not supported (n, m, j_L are packed 10 bits each)"; return KX_ERR_UNSUPPORTED; }
    for (int i = 0; i < N; ++i) {
        if (!(grid->p[i] > 0.0) || !(grid->dp[i] > 0.0) || !isfinite(grid->p[i]) || !isfinite(grid->dp[i]) ||
            (i > 0 && !(grid->p[i] > grid->p[i - 1]))) {
            g_build_err = "grid must have p ascending and > 0, dp > 0";
            return KX_ERR_INVALID_ARG;
        }
    }
    if (!(sp->m >= 0.0) || !(sp->g_chi > 0.0) || !isfinite(sp->m)) { g_build_err = "need m >= 0 and g_chi > 0"; return KX_ERR_INVALID_ARG; }
    if (!isfinite(msq->M2_0) || !isfinite(msq->m_med)) { g_build_err = "non-finite |M|^2 parameters"; return KX_ERR_INVALID_ARG; }
    kx_opts_t o = {KX_INTERP_LOG, KX_STORE_TILED, KX_FP64, KX_EXP_TABLE, 0, 0, 0, 0, 1e-300, 1e-12};
    if (opts) o = *opts;
    if (o.loss_nodes == 0) o.loss_nodes = 24;
    if (o.precision != KX_FP64 && o.precision != KX_FP32) { g_build_err = "unknown precision"; return KX_ERR_INVALID_ARG; }
    if (o.precision == KX_FP32 && o.statistics != KX_STAT_CLASSICAL) {
        g_build_err = "fp32 mode is implemented for classical statistics only";
        return KX_ERR_UNSUPPORTED;
    }
    if (o.storage != KX_STORE_SYM_ROWS && o.storage != KX_STORE_TILED) { g_build_err = "unknown storage mode"; return KX_ERR_UNSUPPORTED; }
    if (o.loss_nodes != 8 && o.loss_nodes != 16 && o.loss_nodes != 24 && o.loss_nodes != 32) {
        g_build_err = "loss_nodes must be 0 (default 24), 8, 16, 24 or 32";
        return KX_ERR_INVALID_ARG;
    }
    if (o.interp != KX_INTERP_LOG && o.interp != KX_INTERP_LINEAR) { g_build_err = "unknown interpolation"; return KX_ERR_INVALID_ARG; }
    if (o.statistics != KX_STAT_CLASSICAL && o.statistics != KX_STAT_BOSE && o.statistics != KX_STAT_FERMI) {
        g_build_err = "statistics must be 0 (classical), +1 (Bose) or -1 (Fermi)";
        return KX_ERR_INVALID_ARG;
    }
    if (o.statistics != KX_STAT_CLASSICAL && o.interp != KX_INTERP_LOG) {
        g_build_err = "quantum statistics need KX_INTERP_LOG (eq. B.20)";
        return KX_ERR_UNSUPPORTED;
    }
    if (o.statistics != KX_STAT_CLASSICAL) o.storage = KX_STORE_SYM_ROWS;     // evaluated by the exact streaming kernel
    if (o.precision == KX_FP32) o.storage = KX_STORE_SYM_ROWS;                // the fp32 contraction is a streaming kernel
    if (o.n_mu < 0 || o.n_mu > 4096 || o.reserved != 0) { g_build_err = "n_mu must be in [0, 4096] and reserved 0"; return KX_ERR_INVALID_ARG; }
    if (o.exp_impl != KX_EXP_TABLE && o.exp_impl != KX_EXP_LIBM) { g_build_err = "unknown exp_impl"; return KX_ERR_INVALID_ARG; }
    if (!(o.f_floor >= 1e-300) || !(o.eps_supp >= 0.0)) { g_build_err = "need f_floor >= 1e-300 and eps_supp >= 0"; return KX_ERR_INVALID_ARG; }

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        g_build_err = "no usable CUDA device (libkx has no CPU fallback)";
        return KX_ERR_CUDA;
    }
    DeviceGuard guard(device);
    if (!guard.ok) { g_build_err = "cudaSetDevice failed"; return KX_ERR_CUDA; }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess || prop.major != 10) {
        g_build_err = "libkx is built for sm_100a (B200) only";
        return KX_ERR_CUDA;
    }

    kx_handle_s* h = new (std::nothrow) kx_handle_s();
    if (!h) { g_build_err = "out of host memory"; return KX_ERR_ALLOC; }
    h->device = device;
    h->p_lo = grid->p[0]; h->p_hi = grid->p[N - 1];
    h->sm_count = prop.multiProcessorCount;
    h->nnz_stale = true;
    h->storage = o.storage;
    KxDev& d = h->d;
    d = KxDev{};
    h->t = KxTiled{};
    d.N = N; d.interp = o.interp; d.exp_impl = o.exp_impl; d.eta = o.statistics; d.chunk = 0; d.prec = o.precision;
    d.m = sp->m; d.g_chi = sp->g_chi; d.M2_0 = msq->M2_0; d.m_med = msq->m_med;
    d.f_floor = o.f_floor; d.eps_supp = o.eps_supp;
    cudaStream_t s = (cudaStream_t)stream;

    auto fail = [&](kx_status_t rc) { g_build_err = h->err; kx_destroy(h); return rc; };
    auto body = [&]() -> kx_status_t {
        // one blob: 8 double arrays [N], exp table, int tables
        const size_t nd = (size_t)8 * N + (1u << KX_EXP_BITS);
        const size_t n2 = (size_t)N * N;
        const size_t bytes = nd * 8 + (n2 * 2 + (n2 + 1) + 2 * (size_t)(N + 1) + 4 + KX_BLUT_MAX + 4) * 4;
        KX_CUDA(cudaMalloc(&h->dev_blob, bytes));
        double* dp_ = (double*)h->dev_blob;
        double* P = dp_;            dp_ += N;
        double* DP = dp_;           dp_ += N;
        d.E = dp_;                  dp_ += N;
        d.K = dp_;                  dp_ += N;
        d.h = dp_;                  dp_ += N;
        d.invdK = dp_;              dp_ += N;
        d.arow = dp_;               dp_ += N;
        d.ccol = dp_;               dp_ += N;
        double* tab = dp_;          dp_ += (1u << KX_EXP_BITS);
        int* ip = (int*)dp_;
        d.run_mlo = ip;             ip += n2;
        d.run_len = ip;             ip += n2;
        d.run_off = (unsigned*)ip;  ip += n2 + 1;
        d.rowptr = (unsigned*)ip;   ip += N + 1;
        d.taskptr = (unsigned*)ip;  ip += N + 1;
        h->flag = ip;               ip += 4;
        d.blut = (unsigned*)ip;
        d.p = P; d.dp = DP; d.exptab = tab;
        std::vector<double> t(1u << KX_EXP_BITS);
        for (unsigned k = 0; k < (1u << KX_EXP_BITS); ++k)
            t[k] = (double)exp2l((long double)k / (long double)(1u << KX_EXP_BITS));
        KX_CUDA(cudaMemcpyAsync(P, grid->p, (size_t)N * 8, cudaMemcpyHostToDevice, s));
        KX_CUDA(cudaMemcpyAsync(DP, grid->dp, (size_t)N * 8, cudaMemcpyHostToDevice, s));
        KX_CUDA(cudaMemcpyAsync(tab, t.data(), t.size() * 8, cudaMemcpyHostToDevice, s));
        KX_CUDA(cudaMemsetAsync(h->flag, 0, 4, s));
        KX_CUDA(cudaMalloc((void**)&h->bar, 16));
        KX_CUDA(cudaMemsetAsync(h->bar, 0, 16, s));
        KX_CUDA(kx_dmma_configure());
        if (o.n_mu > 0) {
            // Gauss-Legendre nodes and weights on [-1,1] (constants, not data dependent): Newton on P_n in long double
            const int n = o.n_mu;
            std::vector<double> gl(2 * (size_t)n);
            const long double pi = 3.14159265358979323846264338327950288L;
            for (int k = 0; k < n; ++k) {
                long double x = cosl(pi * (k + 0.75L) / (n + 0.5L)), dpn = 1.0L;
                for (int it = 0; it < 100; ++it) {
                    long double p0 = 1.0L, p1 = x;
                    for (int j = 2; j <= n; ++j) { long double p2 = ((2 * j - 1) * x * p1 - (j - 1) * p0) / j; p0 = p1; p1 = p2; }
                    if (n == 1) { p0 = 1.0L; p1 = x; }
                    dpn = n * (x * p1 - p0) / (x * x - 1.0L);
                    const long double dx = p1 / dpn;
                    x -= dx;
                    if (fabsl(dx) < 1e-19L) break;
                }
                long double p0 = 1.0L, p1 = x;
                for (int j = 2; j <= n; ++j) { long double p2 = ((2 * j - 1) * x * p1 - (j - 1) * p0) / j; p0 = p1; p1 = p2; }
                dpn = n * (x * p1 - p0) / (x * x - 1.0L);
                gl[n - 1 - k] = (double)x;                                   // ascending
                gl[(size_t)n + n - 1 - k] = (double)(2.0L / ((1.0L - x * x) * dpn * dpn));
            }
            KX_CUDA(cudaMalloc((void**)&h->gl, gl.size() * 8));
            KX_CUDA(cudaMemcpyAsync(h->gl, gl.data(), gl.size() * 8, cudaMemcpyHostToDevice, s));
            KX_CUDA(cudaStreamSynchronize(s));
            d.n_mu = n; d.gl_mu = h->gl; d.gl_w = h->gl + n;
        }
        KX_CUDA(kx_launch_kinematics(d, d.m, s));
        KX_CUDA(kx_launch_runs(d, s));
        unsigned nnz = 0;
        KX_CUDA(cudaMemcpyAsync(&nnz, d.run_off + n2, 4, cudaMemcpyDeviceToHost, s));
        KX_CUDA(cudaStreamSynchronize(s));
        kx_status_t rc = alloc_tensor(h, (long long)nnz);
        if (rc != KX_OK) return rc;
        KX_CUDA(kx_launch_fill(d, s));
        KX_CUDA(cudaStreamSynchronize(s));
        h->nnz = nnz; h->nnz_stale = false; h->chunk_for_B = 0;
        if (h->storage == KX_STORE_TILED) {
            KxTiled& t = h->t;
            t.NT = (N + KX_TI - 1) / KX_TI;
            t.Q = d.interp == KX_INTERP_LOG ? o.loss_nodes : 2;
            t.LC = ((N - 1) * t.Q + 15) / 16;
            t.NR8 = (N + 7) / 8;
            t.RS = (N + 255) / 256;
            // loss operand: fixed size; the padding (k >= (N-1) Q, rows >= N) stays zero for good
            KX_CUDA(dalloc(&t.AL, (size_t)t.LC * t.NR8 * 128));
            KX_CUDA(cudaMemsetAsync(t.AL, 0, (size_t)t.LC * t.NR8 * 128 * 8, s));
            // small tables: trun_mlo, trun_q [NT*N], trun_off [NT*(N+1)], vtptr [NT+1], dct [Q*Q], nodes [Q]
            const size_t tn = (size_t)t.NT * N;
            const size_t ints = tn * 2 + (size_t)t.NT * (N + 1) + (size_t)(t.NT + 1);
            const size_t ints_pad = (ints + 1) & ~(size_t)1;
            KX_CUDA(cudaMalloc(&h->tiled_blob, ints_pad * 4 + ((size_t)t.Q * t.Q + t.Q) * 8));
            int* tp = (int*)h->tiled_blob;
            t.trun_mlo = tp;                 tp += tn;
            t.trun_q = (unsigned*)tp;        tp += tn;
            t.trun_off = (unsigned*)tp;      tp += (size_t)t.NT * (N + 1);
            t.vtptr = (unsigned*)tp;
            double* dd = (double*)((int*)h->tiled_blob + ints_pad);
            t.dct = dd; t.nodes = dd + (size_t)t.Q * t.Q;
            // constants of the discrete Chebyshev transform (not data dependent), in long double
            const int Q = t.Q;
            std::vector<double> tab((size_t)Q * Q + Q);
            const long double pi = 3.14159265358979323846264338327950288L;
            for (int c = 0; c < Q; ++c)
                for (int q = 0; q < Q; ++q)
                    tab[(size_t)c * Q + q] = (double)((c == 0 ? 1.0L : 2.0L) / Q * cosl(c * (2 * q + 1) * pi / (2 * Q)));
            for (int q = 0; q < Q; ++q) tab[(size_t)Q * Q + q] = (double)(0.5L * (1.0L + cosl((2 * q + 1) * pi / (2 * Q))));
            long double lf = 1.0L;           // log2(2 / Q!)
            for (int k = 2; k <= Q; ++k) lf -= log2l((long double)k);
            t.flag_log2 = (double)lf;
            KX_CUDA(cudaMemcpyAsync(dd, tab.data(), tab.size() * 8, cudaMemcpyHostToDevice, s));
            KX_CUDA(cudaStreamSynchronize(s));
            kx_status_t rc2 = build_tiled(h, s);
            if (rc2 != KX_OK) return rc2;
            KX_CUDA(cudaStreamSynchronize(s));
        }
        return KX_OK;
    };
    kx_status_t rc = body();
    if (rc != KX_OK) return fail(rc);
    *out = h;
    return KX_OK;
}

kx_status_t kx_set_mass(kx_handle_t h, double m, void* stream)
{
    if (!h) return KX_ERR_INVALID_ARG;
    if (!(m >= 0.0) || !isfinite(m)) { h->err = "need finite m >= 0"; return KX_ERR_INVALID_ARG; }
    DeviceGuard guard(h->device);
    cudaStream_t s = (cudaStream_t)stream;
    const long long ub = tri_entries(h->d.N);
    if (h->cap < ub) {   // the new mass may keep more triples: size for every (i, n<=m)
        KX_CUDA(cudaStreamSynchronize(s));
        kx_status_t rc = alloc_tensor(h, ub);
        if (rc != KX_OK) return rc;
    }
    return rebuild(h, m, s);
}

kx_status_t kx_collide_ex(kx_handle_t h, const double* f, double* C, double* gain, double* loss,
                          double* diag, int32_t B, uint32_t flags, void* stream)
{
    if (!h) return KX_ERR_INVALID_ARG;
    DeviceGuard guard(h->device);
    return collide_impl(h, f, C, gain, loss, diag, B, flags, (cudaStream_t)stream);
}

kx_status_t kx_collide(kx_handle_t h, const double* f, double* C, int32_t B, uint32_t flags, void* stream)
{
    if (!h) return KX_ERR_INVALID_ARG;
    if (!C) { h->err = "C is NULL"; return KX_ERR_INVALID_ARG; }
    return kx_collide_ex(h, f, C, nullptr, nullptr, nullptr, B, flags, stream);
}

kx_status_t kx_collide_parts(kx_handle_t h, const double* f, double* gain, double* loss, int32_t B, void* stream)
{
    return kx_collide_ex(h, f, nullptr, gain, loss, nullptr, B, 0u, stream);
}

kx_status_t kx_collide_host(kx_handle_t h, const double* f_host, double* C_host, int32_t B,
                            uint32_t flags, void* stream)
{
    if (!h) return KX_ERR_INVALID_ARG;
    if (!f_host || !C_host || B < 1) { h->err = "null host buffer or B < 1"; return KX_ERR_INVALID_ARG; }
    DeviceGuard guard(h->device);
    cudaStream_t s = (cudaStream_t)stream;
    kx_status_t rc = ensure_ws(h, B);
    if (rc != KX_OK) return rc;
    const size_t bn = (size_t)B * h->d.N;
    double* fd = h->hostio;
    double* Cd = h->hostio + (size_t)h->wsB * h->d.N;
    KX_CUDA(cudaMemcpyAsync(fd, f_host, bn * 8, cudaMemcpyHostToDevice, s));
    // A pinned (page-locked, device-mapped) result buffer is written by the finishing phase itself: the stores travel to the
    // host while the kernel runs, and the separate device->host copy with its launch and DMA latency (about 10 us) is gone.
    // Pageable memory takes the staging buffer and a copy.
    double* C_direct = nullptr;
    {
        cudaPointerAttributes at;
        if (cudaPointerGetAttributes(&at, C_host) == cudaSuccess && at.type == cudaMemoryTypeHost && at.devicePointer &&
            ((uintptr_t)at.devicePointer & 15u) == 0)
            C_direct = static_cast<double*>(at.devicePointer);
        else
            (void)cudaGetLastError();        // an unregistered host pointer is not an error here
    }
    rc = collide_impl(h, fd, C_direct ? C_direct : Cd, nullptr, nullptr, nullptr, B, flags, s);
    if (rc != KX_OK) return rc;
    if (!C_direct) KX_CUDA(cudaMemcpyAsync(C_host, Cd, bn * 8, cudaMemcpyDeviceToHost, s));
    KX_CUDA(cudaStreamSynchronize(s));
    return KX_OK;
}

kx_status_t kx_moments(kx_handle_t h, const double* f, int32_t B,
                       double* n, double* rho, double* p1, double* p2, void* stream)
{
    if (!h) return KX_ERR_INVALID_ARG;
    kx_status_t rc = check_batch(h, f, B);
    if (rc != KX_OK) return rc;
    DeviceGuard guard(h->device);
    KX_CUDA(kx_launch_moments(h->d, f, B, n, rho, p1, p2, 1, (cudaStream_t)stream));
    return KX_OK;
}

kx_status_t kx_evolve(kx_handle_t h, double* f, int32_t B, const kx_source_t* src,
                      const kx_evolve_t* ctl, void* stream)
{
    if (!h) return KX_ERR_INVALID_ARG;
    kx_status_t rc = check_batch(h, f, B);
    if (rc != KX_OK) return rc;
    if (!ctl || !ctl->tau || ctl->S < 0) { h->err = "ctl, ctl->tau must be set and S >= 0"; return KX_ERR_INVALID_ARG; }
    if (ctl->method != KX_EULER && ctl->method != KX_HEUN && ctl->method != KX_RK4) { h->err = "unknown method"; return KX_ERR_INVALID_ARG; }
    const int nsrc = src ? src->nsrc : 0;
    if (nsrc < 0 || nsrc > KX_MAX_SRC || (nsrc > 0 && (!src->G || !src->amp))) { h->err = "bad source description"; return KX_ERR_INVALID_ARG; }
    if ((ctl->flags & KX_DIAG) && !ctl->diag) { h->err = "KX_DIAG needs ctl->diag"; return KX_ERR_INVALID_ARG; }
    DeviceGuard guard(h->device);
    cudaStream_t s = (cudaStream_t)stream;
    const int N = h->d.N, S = ctl->S;
    if (ctl->mass && h->cap < tri_entries(N)) {
        KX_CUDA(cudaStreamSynchronize(s));
        if ((rc = alloc_tensor(h, tri_entries(N))) != KX_OK) return rc;
        if ((rc = rebuild(h, h->d.m, s)) != KX_OK) return rc;
    }
    if ((rc = ensure_ws(h, B)) != KX_OK) return rc;
    double* kappa_d = nullptr;
    if (ctl->kappa) {
        kappa_d = h->Cbuf + (size_t)h->wsB * N;
        KX_CUDA(cudaMemcpyAsync(kappa_d, ctl->kappa, (size_t)B * 8, cudaMemcpyHostToDevice, s));
    }
    KX_CUDA(cudaMemsetAsync(h->flag, 0, 4, s));
    const bool diag = (ctl->flags & KX_DIAG) != 0;
    const int nstage = ctl->method == KX_EULER ? 1 : (ctl->method == KX_HEUN ? 2 : 4);
    double kin_mass = h->d.m;        // mass of the kinematics arrays on the device
    double ten_mass = h->d.m;        // mass the tensor was built for
    bool have_yd = false;            // yd already holds the current stage input (written by the last finish)
    // a static tensor is evaluated through the tiled (DMMA) operand; with a mass schedule every stage has new
    // kinematics, and re-deriving the Chebyshev moments per stage costs more than the exact streaming path
    const bool use_tiled = h->storage == KX_STORE_TILED && !ctl->mass && nnz_estimate(h) * B > kSmallProblem;
    if (use_tiled && (rc = ensure_tiled(h, s)) != KX_OK) return rc;

    // Small static-mass problems without per-step diagnostics: the whole integration is ONE cooperative launch
    // (k_stream_run: two grid barriers per stage instead of a launch per stage)
    if (!use_tiled && !ctl->mass && !diag && S > 0 && kx_stream_run_supported(h->d)) {
        const size_t need = (size_t)(S + 1) + (ctl->rate ? (size_t)(2 * S + 1) : 0) + (size_t)nsrc * S;
        if (h->runbuf_cap < need) {
            KX_CUDA(cudaStreamSynchronize(s));
            cudaFree(h->runbuf); h->runbuf = nullptr; h->runbuf_cap = 0;
            KX_CUDA(dalloc(&h->runbuf, need + 1024));
            h->runbuf_cap = need + 1024;
        }
        double* tau_d = h->runbuf;
        double* rate_d = ctl->rate ? tau_d + (S + 1) : nullptr;
        double* amp_d = nsrc ? tau_d + (S + 1) + (ctl->rate ? (2 * S + 1) : 0) : nullptr;
        KX_CUDA(cudaMemcpyAsync(tau_d, ctl->tau, (size_t)(S + 1) * 8, cudaMemcpyHostToDevice, s));
        if (rate_d) KX_CUDA(cudaMemcpyAsync(rate_d, ctl->rate, (size_t)(2 * S + 1) * 8, cudaMemcpyHostToDevice, s));
        if (amp_d) KX_CUDA(cudaMemcpyAsync(amp_d, src->amp, (size_t)nsrc * S * 8, cudaMemcpyHostToDevice, s));
        if ((rc = ensure_tasks(h, B, s)) != KX_OK) return rc;
        KxStage st = {};
        st.flags = ctl->flags & KX_PROJECT;
        st.diag_stride = 6;
        st.evolve = 1; st.rk_method = ctl->method;
        st.kappa = kappa_d;
        st.nsrc = nsrc; st.G = nsrc ? src->G : nullptr;
        st.f = f; st.fstage = h->fstage; st.k1 = h->k1; st.k2 = h->k2; st.k3 = h->k3;
        st.ydnext = h->yd; st.flag = h->flag;
        st.part = h->part; st.bar = h->bar; st.fb_count = h->bar + 2;
        h->epoch += 2; st.epoch = h->epoch;
        st.trace = nullptr;
        KX_CUDA(kx_launch_stream_run(h->d, h->sm_count, f, B, st, ctl->method, S, tau_d, rate_d, amp_d, &h->bar_total, s));
        int flag1 = 0;
        KX_CUDA(cudaMemcpyAsync(&flag1, h->flag, 4, cudaMemcpyDeviceToHost, s));
        KX_CUDA(cudaStreamSynchronize(s));
        if (flag1) { h->err = "kx_evolve: f became non-finite"; return KX_ERR_NONFINITE; }
        return KX_OK;
    }

    for (int k = 0; k < S; ++k) {
        const double dt = ctl->tau[k + 1] - ctl->tau[k];
        for (int stg = 0; stg < nstage; ++stg) {
            // node (0), midpoint (1) or end (2) of the step for this stage
            int pos;
            if (ctl->method == KX_EULER) pos = 0;
            else if (ctl->method == KX_HEUN) pos = stg == 0 ? 0 : 2;
            else pos = stg == 0 ? 0 : (stg == 3 ? 2 : 1);
            const double R = ctl->rate ? ctl->rate[2 * k + pos] : 1.0;
            if (ctl->mass) {
                const double m = ctl->mass[2 * k + pos];
                if (m != ten_mass || m != kin_mass) {
                    if ((rc = rebuild(h, m, s)) != KX_OK) return rc;
                    ten_mass = kin_mass = m;
                }
            }
            if ((rc = ensure_tasks(h, B, s)) != KX_OK) return rc;
            const double* fin = stg == 0 ? f : h->fstage;
            KxStage st = {};
            st.flags = ctl->flags & KX_PROJECT;
            st.diag = (diag && stg == 0) ? ctl->diag + (size_t)k * B * 6 : nullptr;
            st.diag_stride = 6;
            st.evolve = 1; st.rk_method = ctl->method; st.rk_stage = stg;
            st.dt = dt; st.rate = R; st.kappa = kappa_d;
            st.nsrc = nsrc; st.G = nsrc ? src->G : nullptr;
            for (int q = 0; q < nsrc; ++q) st.amp[q] = src->amp[(size_t)q * S + k];
            st.f = f; st.fstage = h->fstage; st.k1 = h->k1; st.k2 = h->k2; st.k3 = h->k3;
            st.ydnext = use_tiled ? nullptr : h->yd; st.flag = h->flag;
            if ((rc = launch_step(h, fin, B, have_yd, use_tiled, &st, s)) != KX_OK) return rc;
            have_yd = !use_tiled;
        }
        if (diag) {
            if (ctl->mass) {
                const double mend = ctl->mass[2 * k + 2];
                if (mend != kin_mass) { KX_CUDA(kx_launch_kinematics(h->d, mend, s)); kin_mass = mend; }
            }
            double* dg = ctl->diag + (size_t)k * B * 6;
            KX_CUDA(kx_launch_moments(h->d, f, B, dg + 4, dg + 5, nullptr, nullptr, 6, s));
        }
    }
    if (ctl->mass && kin_mass != ten_mass) {   // leave the handle consistent
        if ((rc = rebuild(h, kin_mass, s)) != KX_OK) return rc;
    }
    int flag = 0;
    KX_CUDA(cudaMemcpyAsync(&flag, h->flag, 4, cudaMemcpyDeviceToHost, s));
    KX_CUDA(cudaStreamSynchronize(s));
    if (flag) { h->err = "kx_evolve: f became non-finite"; return KX_ERR_NONFINITE; }
    return KX_OK;
}

kx_status_t kx_delta_source(kx_handle_t h, double p0, double* G, void* stream)
{
    if (!h) return KX_ERR_INVALID_ARG;
    if (!G || !(p0 >= h->p_lo && p0 <= h->p_hi)) { h->err = "kx_delta_source: G is NULL or p0 outside the grid"; return KX_ERR_INVALID_ARG; }
    DeviceGuard guard(h->device);
    KX_CUDA(kx_launch_delta_source(h->d, p0, G, (cudaStream_t)stream));
    return KX_OK;
}

kx_status_t kx_evolve_adaptive(kx_handle_t h, double* f, int32_t B, const kx_source_t* src,
                               const kx_adaptive_t* ctl, kx_adaptive_result_t* result, void* stream)
{
    if (!h) return KX_ERR_INVALID_ARG;
    kx_status_t rc = check_batch(h, f, B);
    if (rc != KX_OK) return rc;
    if (!ctl || !(ctl->u1 > ctl->u0) || !(ctl->du0 > 0.0) || !(ctl->rtol >= 0.0) || !(ctl->atol >= 0.0) ||
        !(ctl->rtol + ctl->atol > 0.0) || !(ctl->safety > 0.0 && ctl->safety <= 1.0) || ctl->max_steps < 1 ||
        !isfinite(ctl->rate0) || !isfinite(ctl->rate_slope) || !isfinite(ctl->mass_slope) || !isfinite(ctl->du_fixed) ||
        !isfinite(ctl->eps_switch)) {
        h->err = "kx_evolve_adaptive: need u1 > u0, du0 > 0, rtol, atol >= 0 (not both 0), 0 < safety <= 1, max_steps >= 1, finite rates and slopes";
        return KX_ERR_INVALID_ARG;
    }
    const bool regime1 = ctl->eps_switch > 0.0;
    if (regime1 && !(ctl->du_fixed > 0.0)) { h->err = "kx_evolve_adaptive: eps_switch > 0 needs du_fixed > 0"; return KX_ERR_INVALID_ARG; }
    const int nsrc = (src && ctl->amp) ? src->nsrc : 0;
    if (nsrc < 0 || nsrc > KX_MAX_SRC || (nsrc > 0 && !src->G)) { h->err = "bad source description"; return KX_ERR_INVALID_ARG; }
    DeviceGuard guard(h->device);
    cudaStream_t s = (cudaStream_t)stream;
    const int N = h->d.N;
    const bool mass_var = ctl->mass_slope != 0.0;
    const double mass0 = h->d.m;
    if (mass_var && h->cap < tri_entries(N)) {       // another mass may keep more triples: size for every (i, n <= m)
        KX_CUDA(cudaStreamSynchronize(s));
        if ((rc = alloc_tensor(h, tri_entries(N))) != KX_OK) return rc;
        if ((rc = rebuild(h, h->d.m, s)) != KX_OK) return rc;
    }
    if ((rc = ensure_ws(h, B)) != KX_OK) return rc;
    if (!h->adapt) KX_CUDA(cudaMalloc((void**)&h->adapt, sizeof(KxAdapt) + 64 + KX_MAX_SRC * 8));
    double* m_dev = reinterpret_cast<double*>(reinterpret_cast<char*>(h->adapt) + ((sizeof(KxAdapt) + 15) & ~(size_t)15));
    double* amp_dev = m_dev + 2;
    double* kappa_d = nullptr;
    if (ctl->kappa) {
        kappa_d = h->Cbuf + (size_t)h->wsB * N;
        KX_CUDA(cudaMemcpyAsync(kappa_d, ctl->kappa, (size_t)B * 8, cudaMemcpyHostToDevice, s));
    }
    if (nsrc > 0) KX_CUDA(cudaMemcpyAsync(amp_dev, ctl->amp, (size_t)nsrc * 8, cudaMemcpyHostToDevice, s));
    KxAdapt init = {};
    init.u = ctl->u0;
    init.du = ctl->du0 < ctl->u1 - ctl->u0 ? ctl->du0 : ctl->u1 - ctl->u0;
    init.errkey = 0;                 // key of +0.0
    init.switched = regime1 ? 0 : 1;
    init.u_switch = regime1 ? ctl->u1 : ctl->u0;
    KX_CUDA(cudaMemcpyAsync(h->adapt, &init, sizeof init, cudaMemcpyHostToDevice, s));
    KX_CUDA(cudaMemsetAsync(h->flag, 0, 4, s));
    // with m(u) every stage has new kinematics: the exact streaming path (as kx_evolve with a mass schedule)
    const bool use_tiled = h->storage == KX_STORE_TILED && !mass_var && nnz_estimate(h) * B > kSmallProblem;
    if (use_tiled && (rc = ensure_tiled(h, s)) != KX_OK) return rc;
    if ((rc = ensure_tasks(h, B, s)) != KX_OK) return rc;

    // a1-a3 for m(u_stage), u_stage read from the controller state on the device
    auto rebuild_at = [&](int stage) -> kx_status_t {
        KX_CUDA(kx_launch_adapt_mass(h->adapt, stage, ctl->u0, mass0, ctl->mass_slope, m_dev, s));
        h->d.m_dev = m_dev;
        KX_CUDA(kx_launch_kinematics(h->d, 0.0, s));
        KX_CUDA(kx_launch_runs(h->d, s));
        KX_CUDA(kx_launch_fill(h->d, s));
        h->nnz_stale = true; h->chunk_for_B = 0; h->tiled_ok = false;
        return ensure_tasks(h, B, s);
    };
    auto finish = [&](kx_status_t code) -> kx_status_t {      // leave the handle with a host-side mass again
        if (mass_var) {
            h->d.m_dev = nullptr;
            KxAdapt st2 = {};
            if (cudaMemcpyAsync(&st2, h->adapt, sizeof st2, cudaMemcpyDeviceToHost, s) == cudaSuccess &&
                cudaStreamSynchronize(s) == cudaSuccess) {
                const kx_status_t r2 = rebuild(h, mass0 * exp(ctl->mass_slope * (st2.u - ctl->u0)), s);
                if (code == KX_OK && r2 != KX_OK) code = r2;
            }
        }
        return code;
    };

    KxAdapt state = init;
    // ---- regime 1: sources only on fixed intervals, Gamma_2->2/H monitored at every interval boundary
    while (regime1 && !state.switched && !state.done) {
        for (int a = 0; a < 8; ++a) {
            if (mass_var && (rc = rebuild_at(0)) != KX_OK) return finish(rc);
            KxStage st = {};
            st.loss = h->k3; st.diag_stride = 4; st.evolve = 0;
            if ((rc = launch_step(h, f, B, false, use_tiled, &st, s)) != KX_OK) return finish(rc);
            KX_CUDA(kx_launch_regime1_step(h->d, f, h->k3, B, kappa_d, nsrc, nsrc ? src->G : nullptr, amp_dev, h->adapt,
                                           ctl->u0, ctl->u1, ctl->du_fixed, ctl->eps_switch, ctl->rate0, ctl->rate_slope, s));
        }
        KX_CUDA(cudaMemcpyAsync(&state, h->adapt, sizeof state, cudaMemcpyDeviceToHost, s));
        KX_CUDA(cudaStreamSynchronize(s));
    }
    // ---- regime 2: adaptive Heun from the switch point
    if (regime1 && state.switched && !state.done) {
        state.du = ctl->du0 < ctl->u1 - state.u ? ctl->du0 : ctl->u1 - state.u;
        state.errkey = 0;
        KX_CUDA(cudaMemcpyAsync(h->adapt, &state, sizeof state, cudaMemcpyHostToDevice, s));
    }
    int attempts = 0;
    while (attempts < ctl->max_steps && !state.done) {
        const int chunk = ctl->max_steps - attempts < 8 ? ctl->max_steps - attempts : 8;
        for (int a = 0; a < chunk; ++a) {
            for (int stg = 0; stg < 2; ++stg) {
                if (mass_var && (rc = rebuild_at(stg)) != KX_OK) return finish(rc);
                const double* fin = stg == 0 ? f : h->fstage;
                KxStage st = {};
                st.flags = ctl->flags & KX_PROJECT;
                st.diag_stride = 6;
                st.evolve = 1; st.rk_method = KX_HEUN_ADAPT; st.rk_stage = stg;
                st.kappa = kappa_d;
                st.nsrc = nsrc; st.G = nsrc ? src->G : nullptr;
                for (int q = 0; q < nsrc; ++q) st.amp[q] = ctl->amp[q];
                st.f = f; st.fstage = h->fstage; st.k1 = h->k1; st.k2 = h->k2; st.k3 = h->k3;
                st.ydnext = (!use_tiled && stg == 0) ? h->yd : nullptr;
                st.flag = h->flag;
                st.ad = h->adapt; st.ad_u0 = ctl->u0; st.ad_rate0 = ctl->rate0; st.ad_slope = ctl->rate_slope;
                st.ad_rtol = ctl->rtol; st.ad_atol = ctl->atol;
                if ((rc = launch_step(h, fin, B, /*have_yd=*/stg == 1 && !use_tiled, use_tiled, &st, s)) != KX_OK) return finish(rc);
            }
            KX_CUDA(kx_launch_adapt_step(h->d, f, h->k2, B, h->adapt, ctl->u1, ctl->safety, h->flag, s));
        }
        attempts += chunk;
        KX_CUDA(cudaMemcpyAsync(&state, h->adapt, sizeof state, cudaMemcpyDeviceToHost, s));
        KX_CUDA(cudaStreamSynchronize(s));
    }
    int flag = 0;
    KX_CUDA(cudaMemcpyAsync(&flag, h->flag, 4, cudaMemcpyDeviceToHost, s));
    KX_CUDA(cudaStreamSynchronize(s));
    if (result) {
        result->u = state.u; result->du = state.du;
        result->accepted = state.accepted; result->rejected = state.rejected; result->done = state.done;
        result->switched = state.switched; result->u_switch = state.u_switch; result->fixed_steps = state.fixed_steps;
        result->ratio = state.ratio;
    }
    rc = finish(KX_OK);
    if (rc != KX_OK) return rc;
    if (flag) { h->err = "kx_evolve_adaptive: f became non-finite"; return KX_ERR_NONFINITE; }
    return KX_OK;
}

kx_status_t kx_reserve(kx_handle_t h, int32_t B, void* stream)
{
    if (!h) return KX_ERR_INVALID_ARG;
    if (B < 1) { h->err = "kx_reserve: B < 1"; return KX_ERR_INVALID_ARG; }
    DeviceGuard guard(h->device);
    cudaStream_t s = (cudaStream_t)stream;
    kx_status_t rc = ensure_ws(h, B);
    if (rc != KX_OK) return rc;
    if ((rc = ensure_tasks(h, B, s)) != KX_OK) return rc;
    if ((rc = ensure_tiled(h, s)) != KX_OK) return rc;
    if (h->storage == KX_STORE_TILED && h->plan_B != B) {
        kx_dmma_plan(h->d, h->t, h->sm_count, h->vt_host.data(), B, &h->plan);
        h->plan_B = B;
    }
    return KX_OK;
}

kx_status_t kx_fallback_members(kx_handle_t h, int64_t* count)
{
    if (!h || !count) return KX_ERR_INVALID_ARG;
    DeviceGuard guard(h->device);
    KX_CUDA(cudaDeviceSynchronize());
    unsigned v = 0;
    KX_CUDA(cudaMemcpy(&v, h->bar + 2, 4, cudaMemcpyDeviceToHost));
    KX_CUDA(cudaMemset(h->bar + 2, 0, 4));
    *count = (int64_t)v;
    return KX_OK;
}

kx_status_t kx_trace(kx_handle_t h, int32_t enable)
{
    if (!h) return KX_ERR_INVALID_ARG;
    DeviceGuard guard(h->device);
    if (enable && !h->trace) {
        KX_CUDA(cudaMalloc((void**)&h->trace, (size_t)KX_TRACE_CTAS * KX_TRACE_SLOTS * 8));
        KX_CUDA(cudaMemset(h->trace, 0, (size_t)KX_TRACE_CTAS * KX_TRACE_SLOTS * 8));
    }
    h->tracing = enable != 0;
    return KX_OK;
}

kx_status_t kx_trace_read(kx_handle_t h, uint64_t* stamps)
{
    if (!h || !stamps) return KX_ERR_INVALID_ARG;
    if (!h->trace) { h->err = "kx_trace_read: tracing was never enabled"; return KX_ERR_INVALID_ARG; }
    DeviceGuard guard(h->device);
    KX_CUDA(cudaDeviceSynchronize());
    KX_CUDA(cudaMemcpy(stamps, h->trace, (size_t)KX_TRACE_CTAS * KX_TRACE_SLOTS * 8, cudaMemcpyDeviceToHost));
    KX_CUDA(cudaMemset(h->trace, 0, (size_t)KX_TRACE_CTAS * KX_TRACE_SLOTS * 8));
    return KX_OK;
}

kx_status_t kx_profile(kx_handle_t h, int32_t enable)
{
    if (!h) return KX_ERR_INVALID_ARG;
    h->profiling = enable != 0;
    return KX_OK;
}

kx_status_t kx_profile_read(kx_handle_t h, double* contract_ms, int64_t* launches)
{
    if (!h) return KX_ERR_INVALID_ARG;
    DeviceGuard guard(h->device);
    KX_CUDA(cudaDeviceSynchronize());
    double sum = 0.0;
    for (size_t k = 0; k < h->prof_used; ++k) {
        float ms = 0.f;
        KX_CUDA(cudaEventElapsedTime(&ms, h->prof_events[k].first, h->prof_events[k].second));
        sum += ms;
    }
    if (contract_ms) *contract_ms = sum;
    if (launches) *launches = (int64_t)h->prof_used;
    h->prof_used = 0;
    return KX_OK;
}

kx_status_t kx_info(kx_handle_t h, int64_t* nnz, int64_t* tensor_bytes, int32_t* n)
{
    if (!h) return KX_ERR_INVALID_ARG;
    DeviceGuard guard(h->device);
    KX_CUDA(cudaDeviceSynchronize());
    if (h->nnz_stale) {
        unsigned v = 0;
        KX_CUDA(cudaMemcpy(&v, h->d.run_off + (size_t)h->d.N * h->d.N, 4, cudaMemcpyDeviceToHost));
        h->nnz = v; h->nnz_stale = false;
    }
    if (nnz) *nnz = h->nnz;
    if (tensor_bytes) {
        if (h->storage == KX_STORE_TILED && h->tiled_ok)
            *tensor_bytes = h->groups * (KX_GROUP_DBL * 8 + 16) + (long long)h->t.LC * h->t.NR8 * 1024;
        else *tensor_bytes = h->nnz * 20;            // W 8 + omega 8 + n|m|j 4
    }
    if (n) *n = h->d.N;
    return KX_OK;
}

kx_status_t kx_tensor_export(kx_handle_t h, int64_t cap, int64_t* rowptr, double* W, double* omega, uint32_t* nmj)
{
    if (!h) return KX_ERR_INVALID_ARG;
    int64_t nnz = 0;
    kx_status_t rc = kx_info(h, &nnz, nullptr, nullptr);
    if (rc != KX_OK) return rc;
    if (cap < nnz) { h->err = "kx_tensor_export: capacity below nnz"; return KX_ERR_INVALID_ARG; }
    DeviceGuard guard(h->device);
    const int N = h->d.N;
    if (rowptr) {
        std::vector<unsigned> rp(N + 1);
        KX_CUDA(cudaMemcpy(rp.data(), h->d.rowptr, (size_t)(N + 1) * 4, cudaMemcpyDeviceToHost));
        for (int i = 0; i <= N; ++i) rowptr[i] = rp[i];
    }
    if (W) KX_CUDA(cudaMemcpy(W, h->d.W, (size_t)nnz * 8, cudaMemcpyDeviceToHost));
    if (omega) KX_CUDA(cudaMemcpy(omega, h->d.omega, (size_t)nnz * 8, cudaMemcpyDeviceToHost));
    if (nmj) KX_CUDA(cudaMemcpy(nmj, h->d.nmj, (size_t)nnz * 4, cudaMemcpyDeviceToHost));
    return KX_OK;
}

kx_status_t kx_kinematics_export(kx_handle_t h, double* E, double* K, double* hw)
{
    if (!h) return KX_ERR_INVALID_ARG;
    DeviceGuard guard(h->device);
    KX_CUDA(cudaDeviceSynchronize());
    const size_t b = (size_t)h->d.N * 8;
    if (E) KX_CUDA(cudaMemcpy(E, h->d.E, b, cudaMemcpyDeviceToHost));
    if (K) KX_CUDA(cudaMemcpy(K, h->d.K, b, cudaMemcpyDeviceToHost));
    if (hw) KX_CUDA(cudaMemcpy(hw, h->d.h, b, cudaMemcpyDeviceToHost));
    return KX_OK;
}

}  // extern "C"
