// kx_contract.cu -- steps a4-a9: gain/loss contraction, raw operator, projection, fused RK stage, moments.
//
//   a4  gain_i = sum_{n<=m} Wsym[i,nm] f_n f_m                              eq. 4.6 with 2.6
//   a5  nu_i   = sum_{n<=m} Wsym[i,nm] f_j~,  loss_i = f_i nu_i
//       LOG:    f_j~ = 2^(y_L + omega_R (y_R - y_L)),  y = log2 max(f, f_floor)   eq. B.20 at eta=0, D7/D8
//       LINEAR: f_j~ = f_L + omega_R (f_R - f_L)                                  eq. B.19
//   a6  C_raw = gain - f_i nu_i
//   a7  projection C.2-C.8 in the basis {1, K_i} (same span as {1, E_i}, well conditioned), diag C.1, C.9
//   a8  Runge-Kutta stage update fused into the finishing kernel                   eq. 4.9
//   a9  moments                                                                    eq. B.2
//
// Work decomposition of the contraction: row i of the row-compressed tensor is cut into tasks of `chunk`
// entries; a persistent CTA loops over tasks, each thread owns entries e0+tid, e0+tid+256, ... and keeps
// BT gain and BT loss accumulators (one per batch member of its group) in registers; a fixed-order
// shuffle/shared-memory reduction writes one partial per (task, b); the finishing kernel adds the
// partials of a row in task order.  No atomics: results are bit-reproducible.
//
// Compiled with --fmad=false; every fused multiply-add below is an explicit fma().
#include "kx_internal.cuh"

namespace {

// ---------------------------------------------------------------- prep: (y_j, y_{j+1}-y_j) per (b, j)
// y of eq. B.20 in base 2: log2(f / (1 + eta f)), f floored (reading D8); LINEAR interpolation works on f itself
__device__ __forceinline__ double kx_yval(double f, int interp, double f_floor, int eta)
{
    if (interp != KX_INTERP_LOG) return f;
    const double ff = fmax(f, f_floor);
    return eta == 0 ? log2(ff) : log2(ff / (1.0 + (double)eta * ff));
}

__global__ void k_prep(KxDev d, const double* __restrict__ f, double2* __restrict__ yd, int B)
{
    int j = blockIdx.x * blockDim.x + threadIdx.x;
    int b = blockIdx.y;
    if (j >= d.N) return;
    const double* fb = f + (size_t)b * d.N;
    double y0 = kx_yval(fb[j], d.interp, d.f_floor, d.eta);
    double y1 = (j + 1 < d.N) ? kx_yval(fb[j + 1], d.interp, d.f_floor, d.eta) : y0;
    yd[(size_t)b * d.N + j] = make_double2(y0, y1 - y0);
}

// ---------------------------------------------------------------- contraction
enum { MODE_LOG_TAB = 0, MODE_LOG_LIBM = 1, MODE_LINEAR = 2 };

// QS = 1: quantum statistics (eq. 4.3).  With x = f_j~ = e^y / (1 - eta e^y) four sums per (row, member) are kept,
//   G1 = sum W f_n f_m,  L1 = sum W x,  G2 = sum W f_n f_m x,  L2 = sum W x (f_n + f_m),
// from which  gain = (1 + eta f_i)(G1 + eta G2),  loss = f_i (L1 + eta L2 + G2)   (eta^2 = 1; k_finish).
template <int BT, int MODE, int QS>
__global__ void __launch_bounds__(KX_CTA, 2)
k_contract(KxDev d, const double* __restrict__ f, const double2* __restrict__ yd,
           double* __restrict__ part, int B, const long long* __restrict__ mstat)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = d.N;
    double2* s_yd = reinterpret_cast<double2*>(smem_raw);                 // [BT][N]
    double* s_f = reinterpret_cast<double*>(s_yd + (size_t)BT * N);       // [BT][N]
    constexpr int NV = QS ? 4 : 2;                                         // sums per (row, member)
    double* s_red = s_f + (size_t)BT * N;                                 // [8][NV*BT]
    double* s_tab = s_red + (KX_CTA / 32) * NV * BT;                       // [256][16] (MODE_LOG_TAB)
    unsigned* s_tp = reinterpret_cast<unsigned*>(s_tab + (MODE == MODE_LOG_TAB ? (KX_EXP_REP << KX_EXP_BITS) : 0)); // [N+1]

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int b0 = blockIdx.y * BT;
    const int nb = min(BT, B - b0);
    kx_pdl_trigger();
    kx_pdl_wait();
    if (mstat) {          // tiled path: only member groups holding a flagged member take the exact streaming path
        // one member per thread and one vote: a single round trip to the statistics instead of one per member
        const int any = __syncthreads_or(tid < nb && kx_member_flagged(mstat, b0 + tid));
        if (!any) return;
    }

    for (int k = tid; k < BT * N; k += KX_CTA) {
        int b = k / N, j = k - b * N;
        if (b < nb) {
            const double fv = f[(size_t)(b0 + b) * N + j];
            if (yd) s_yd[k] = yd[(size_t)(b0 + b) * N + j];
            else {        // fallback of the tiled path: no prepared y, computed here (k_prep's arithmetic)
                const double y0 = kx_yval(fv, d.interp, d.f_floor, d.eta);
                const double y1 = j + 1 < N ? kx_yval(f[(size_t)(b0 + b) * N + j + 1], d.interp, d.f_floor, d.eta) : y0;
                s_yd[k] = make_double2(y0, y1 - y0);
            }
            s_f[k] = fv;
        } else {                                  // ragged last group: harmless values, results discarded
            s_yd[k] = make_double2(0.0, 0.0);
            s_f[k] = 0.0;
        }
    }
    if (MODE == MODE_LOG_TAB)
        for (int k = tid; k < (KX_EXP_REP << KX_EXP_BITS); k += KX_CTA) s_tab[k] = d.exptab[k / KX_EXP_REP];
    for (int k = tid; k <= N; k += KX_CTA) s_tp[k] = d.taskptr[k];
    __syncthreads();

    const unsigned ntasks = s_tp[N];
    const double* tab_lane = s_tab + (lane & (KX_EXP_REP - 1));
    const unsigned chunk = (unsigned)d.chunk;

    for (unsigned task = blockIdx.x; task < ntasks; task += gridDim.x) {
        // row of this task: largest i with taskptr[i] <= task
        int lo = 0, hi = N - 1;
        while (lo < hi) {
            int mid = (lo + hi + 1) >> 1;
            if (s_tp[mid] <= task) lo = mid; else hi = mid - 1;
        }
        const int i = lo;
        const unsigned r0 = d.rowptr[i], r1 = d.rowptr[i + 1];
        const unsigned e0 = r0 + (task - s_tp[i]) * chunk;
        const unsigned e1 = min(e0 + chunk, r1);

        double g[BT], l[BT], g2[QS ? BT : 1], l2[QS ? BT : 1];
#pragma unroll
        for (int b = 0; b < BT; ++b) { g[b] = 0.0; l[b] = 0.0; if (QS) { g2[b] = 0.0; l2[b] = 0.0; } }
        const double eta = (double)d.eta;

        unsigned e = e0 + tid;
        double W = 0.0, om = 0.0;
        unsigned pk = 0;
        if (e < e1) { W = d.W[e]; om = d.omega[e]; pk = d.nmj[e]; }
        while (e < e1) {
            const double Wc = W, omc = om;
            const unsigned pkc = pk;
            e += KX_CTA;
            if (e < e1) { W = d.W[e]; om = d.omega[e]; pk = d.nmj[e]; }   // prefetch the next entry
            const int n = pkc & 1023, m = (pkc >> 10) & 1023, j = pkc >> 20;
#pragma unroll
            for (int b = 0; b < BT; ++b) {
                const double fn = s_f[b * N + n], fm = s_f[b * N + m];
                const double pn = fn * fm;
                g[b] = fma(Wc, pn, g[b]);
                const double2 y = s_yd[b * N + j];
                const double t = fma(omc, y.y, y.x);
                double x;
                if (MODE == MODE_LOG_TAB) x = kx_exp2_tab<KX_EXP_REP>(t, tab_lane);
                else if (MODE == MODE_LOG_LIBM) x = exp2(t);
                else x = t;
                if (QS) {
                    // W f_j~, eq. B.20: x / (1 - eta x) with the reciprocal from the hardware estimate (2^-23) and two
                    // Newton steps (2^-46, 2^-92: full double precision) instead of the IEEE division sequence
                    const double dn = fma(-eta, x, 1.0);
                    double rc;
                    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(rc) : "d"(dn));
                    double er = fma(-dn, rc, 1.0);
                    rc = fma(rc, er, rc);
                    er = fma(-dn, rc, 1.0);
                    rc = fma(rc, er, rc);
                    const double wf = Wc * (x * rc);
                    l[b] += wf;
                    g2[b] = fma(wf, pn, g2[b]);
                    l2[b] = fma(wf, fn + fm, l2[b]);
                } else {
                    l[b] = fma(Wc, x, l[b]);
                }
            }
        }
        // fixed-order reduction: xor butterfly inside the warp, then warps 0..7 in order
#pragma unroll
        for (int b = 0; b < BT; ++b) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                g[b] += __shfl_xor_sync(0xffffffffu, g[b], o);
                l[b] += __shfl_xor_sync(0xffffffffu, l[b], o);
                if (QS) {
                    g2[b] += __shfl_xor_sync(0xffffffffu, g2[b], o);
                    l2[b] += __shfl_xor_sync(0xffffffffu, l2[b], o);
                }
            }
        }
        if (lane == 0) {
#pragma unroll
            for (int b = 0; b < BT; ++b) {
                s_red[warp * NV * BT + NV * b] = g[b];
                s_red[warp * NV * BT + NV * b + 1] = l[b];
                if (QS) { s_red[warp * NV * BT + NV * b + 2] = g2[b]; s_red[warp * NV * BT + NV * b + 3] = l2[b]; }
            }
        }
        __syncthreads();
        if (tid < NV * BT) {
            double acc = 0.0;
#pragma unroll
            for (int w = 0; w < KX_CTA / 32; ++w) acc += s_red[w * NV * BT + tid];
            const int b = tid / NV;
            if (b < nb) part[((size_t)task * B + (b0 + b)) * NV + (tid % NV)] = acc;
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------- block reductions (256 threads, fixed order)
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double* s_red /* [NV*8] */)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < NV; ++k)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_xor_sync(0xffffffffu, v[k], o);
    __syncthreads();
    if (lane == 0)
#pragma unroll
        for (int k = 0; k < NV; ++k) s_red[k * 8 + warp] = v[k];
    __syncthreads();
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        double a = 0.0;
#pragma unroll
        for (int w = 0; w < 8; ++w) a += s_red[k * 8 + w];
        v[k] = a;
    }
}

__device__ __forceinline__ double block_max(double v, double* s_red)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    __syncthreads();
    if (lane == 0) s_red[warp] = v;
    __syncthreads();
    double a = s_red[0];
#pragma unroll
    for (int w = 1; w < 8; ++w) a = fmax(a, s_red[w]);
    return a;
}

// ---------------------------------------------------------------- partials of the DMMA kernel -> (gain, nu)[b, i]
// gain: tile = i/16, groups [a0,a1) of the tile were taken by the gain workers c0..c1 (equal ranges of the Gtot
// groups), slot = c + tile.  loss: supertile = i/256, chunk units [sp LC, (sp+1) LC) of the RS LC units were taken by
// the loss CTAs c0..c1, slot = c + sp.  A CTA adds the partials of 16 rows x 2 members; the slots of an output are
// dealt to 8 threads (slot = first + part, step 8) and the 8 sums are added in part order: a fixed order,
// bit-reproducible.
__global__ void __launch_bounds__(256) k_reduce(int N, int B, KxStage st)
{
    __shared__ double s_g[8][32], s_l[8][32];
    kx_pdl_trigger();
    const int tid = threadIdx.x, part = tid >> 5, o = tid & 31, il = o & 15, bl = o >> 4;
    const int tile = blockIdx.x, b = blockIdx.y * 2 + bl, i = tile * 16 + il;
    const bool on = b < B && i < N;
    // everything that does not depend on the contraction kernel happens before the wait: the slot ranges
    unsigned c0 = 1, c1 = 0, d0 = 1, d1 = 0;
    const double* src = nullptr;
    const double* srl = nullptr;
    if (on) {
        const unsigned Gtot = st.vtptr[st.NT];
        const unsigned a0 = st.vtptr[tile], a1 = st.vtptr[tile + 1];
        if (a1 > a0) {
            c0 = (unsigned)((((unsigned long long)a0 + 1ull) * (unsigned)st.GW - 1ull) / Gtot);
            c1 = (unsigned)(((unsigned long long)a1 * (unsigned)st.GW - 1ull) / Gtot);
        }
        src = st.gpart + ((size_t)tile * st.xstride + b) * 16 + il;
        const unsigned U = (unsigned)st.RS * (unsigned)st.LC;
        const unsigned sp = (unsigned)i >> 8;
        const unsigned l0 = sp * (unsigned)st.LC, l1 = l0 + (unsigned)st.LC;
        d0 = (unsigned)((((unsigned long long)l0 + 1ull) * (unsigned)st.GL - 1ull) / U);
        d1 = (unsigned)(((unsigned long long)l1 * (unsigned)st.GL - 1ull) / U);
        srl = st.lpart + ((size_t)sp * st.xstride + b) * 256 + (i & 255);
    }
    kx_pdl_wait();
    double g = 0.0, nu = 0.0;
    if (on) {
        // all loads of an output are in flight together: the first 8 loss partials are requested before the gain loop
        double vl[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const unsigned c = d0 + part + 8u * (unsigned)u;
            vl[u] = c <= d1 ? srl[(size_t)c * st.xstride * 256] : 0.0;
        }
#pragma unroll 8
        for (unsigned c = c0 + part; c <= c1; c += 8) g += src[(size_t)c * st.xstride * 16];
#pragma unroll
        for (int u = 0; u < 8; ++u) nu += vl[u];
        for (unsigned c = d0 + part + 64u; c <= d1; c += 8) nu += srl[(size_t)c * st.xstride * 256];
    }
    s_g[part][o] = g;
    s_l[part][o] = nu;
    __syncthreads();
    if (part == 0 && on) {
        double G = s_g[0][o], L = s_l[0][o];
#pragma unroll
        for (int k = 1; k < 8; ++k) { G += s_g[k][o]; L += s_l[k][o]; }
        st.gn[(size_t)b * N + i] = make_double2(G, L);
    }
}

// ---------------------------------------------------------------- finishing kernel: one CTA per member b
constexpr int kMaxPerThread = KX_MAX_N / KX_CTA;   // 4

__global__ void __launch_bounds__(KX_CTA)
k_finish(KxDev d, const double* __restrict__ fin, const double* __restrict__ part, int B, KxStage st)
{
    __shared__ double s_red[8 * 8];
    __shared__ double s_y[KX_MAX_N];
    const int N = d.N, tid = threadIdx.x, b = blockIdx.x;
    const double* fb = fin + (size_t)b * N;
    // inputs that no kernel of this call writes (the stage input, the kinematics) are fetched before the wait
    double C[kMaxPerThread], fi[kMaxPerThread], hi_[kMaxPerThread], Ei[kMaxPerThread], Ki[kMaxPerThread];
#pragma unroll
    for (int q = 0; q < kMaxPerThread; ++q) {
        const int i = tid + q * KX_CTA;
        C[q] = 0.0; fi[q] = 0.0; hi_[q] = 0.0; Ei[q] = 0.0; Ki[q] = 0.0;
        if (i < N) { fi[q] = fb[i]; hi_[q] = d.h[i]; Ei[q] = d.E[i]; Ki[q] = d.K[i]; }
    }
    kx_pdl_wait();
    const bool tiled = st.gpart != nullptr && !(st.mstat && kx_member_flagged(st.mstat, b));
    if (st.mstat) {          // last reader of the member's statistics: reset them for the next call
        __syncthreads();
        if (tid == 0) { st.mstat[2 * b] = KX_MSTAT_NONE; st.mstat[2 * b + 1] = 0; }
    }

#pragma unroll
    for (int q = 0; q < kMaxPerThread; ++q) {
        const int i = tid + q * KX_CTA;
        if (i < N) {
            double g = 0.0, nu = 0.0, gq2 = 0.0, lq2 = 0.0;
            if (tiled) {
                const double2 v = st.gn[(size_t)b * N + i];          // partials of the DMMA kernel, added by k_reduce
                g = v.x; nu = v.y;
            } else {
                const unsigned t0 = d.taskptr[i], t1 = d.taskptr[i + 1];
                const int nv = d.eta ? 4 : 2;
                for (unsigned t = t0; t < t1; ++t) {
                    const double* pp = part + ((size_t)t * B + b) * nv;
                    g += pp[0];
                    nu += pp[1];
                    if (d.eta) { gq2 += pp[2]; lq2 += pp[3]; }
                }
            }
            if (d.eta) {                                          // eq. 4.3 from the four sums (see k_contract)
                const double eta = (double)d.eta;
                g = (1.0 + eta * fi[q]) * (g + eta * gq2);
                nu = nu + eta * lq2 + gq2;
            }
            C[q] = fma(-fi[q], nu, g);                            // a6
            if (st.gain) st.gain[(size_t)b * N + i] = g;
            if (st.loss) st.loss[(size_t)b * N + i] = fi[q] * nu;
        }
    }

    const bool project = (st.flags & KX_PROJECT) != 0;
    if (project || st.diag) {
        // C.2 and the denominators of C.1 / C.9
        double v[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
        double fm = 0.0;
#pragma unroll
        for (int q = 0; q < kMaxPerThread; ++q) {
            const double hc = hi_[q] * C[q];
            v[0] += hc;                       // R0 = sum h C
            v[1] += hc * Ki[q];               // RK = sum h K C
            v[2] += hc * Ei[q];               // R1 = sum h E C
            v[3] += fabs(hc);                 // S0
            v[4] += fabs(hc) * Ei[q];         // S1
            fm = fmax(fm, fabs(fi[q]));
        }
        block_sum<5>(v, s_red);
        const double fmax_ = block_max(fm, s_red);
        const double R0 = v[0], RK = v[1], R1 = v[2], S0 = v[3], S1 = v[4];
        double alpha = 0.0, beta = 0.0, D0 = 0.0, D1 = 0.0;
        if (project) {
            double xi[kMaxPerThread];
            double a[3] = {0.0, 0.0, 0.0};
#pragma unroll
            for (int q = 0; q < kMaxPerThread; ++q) {
                const double r = fmax_ > 0.0 ? fabs(fi[q]) / fmax_ : 0.0;     // C.4
                xi[q] = r > d.eps_supp ? r : 0.0;
                const double hx = hi_[q] * xi[q];
                a[0] += hx;                   // A00
                a[1] += hx * Ki[q];           // A0K
                a[2] += hx * Ki[q] * Ki[q];   // AKK
            }
            block_sum<3>(a, s_red);
            const double A00 = a[0], A0K = a[1], AKK = a[2];
            if (fmax_ > 0.0 && A00 > 0.0) {
                const double det = A00 * AKK - A0K * A0K;                    // C.8
                if (det <= 1e-14 * A00 * AKK) { alpha = R0 / A00; beta = 0.0; }   // D9
                else { alpha = (R0 * AKK - RK * A0K) / det; beta = (RK * A00 - R0 * A0K) / det; }
            }
            double dsum[2] = {0.0, 0.0};
#pragma unroll
            for (int q = 0; q < kMaxPerThread; ++q) {
                const double corr = xi[q] * (alpha + beta * Ki[q]);
                C[q] = C[q] - corr;                                          // C.3
                dsum[0] += hi_[q] * fabs(corr);
                dsum[1] += hi_[q] * Ei[q] * fabs(corr);
            }
            if (st.diag) { block_sum<2>(dsum, s_red); D0 = dsum[0]; D1 = dsum[1]; }
        }
        if (st.diag && tid == 0) {
            double* dg = st.diag + (size_t)b * st.diag_stride;
            dg[0] = S0 > 0.0 ? R0 / S0 : 0.0;       // eps_N, C.1
            dg[1] = S1 > 0.0 ? R1 / S1 : 0.0;       // eps_E
            dg[2] = S0 > 0.0 ? D0 / S0 : 0.0;       // R_N, C.9
            dg[3] = S1 > 0.0 ? D1 / S1 : 0.0;       // R_E
        }
    }

    if (st.C) {
#pragma unroll
        for (int q = 0; q < kMaxPerThread; ++q) {
            const int i = tid + q * KX_CTA;
            if (i < N) st.C[(size_t)b * N + i] = C[q];
        }
    }
    if (!st.evolve) return;

    // ---- a8: k = kappa_b R C + sum_s amp_s G_s, then the Runge-Kutta bookkeeping of this stage
    double rate = st.rate, dt = st.dt;
    if (st.rk_method == KX_HEUN_ADAPT) {      // step and rate from the device controller (kx_evolve_adaptive)
        const double u = st.ad->u;
        dt = st.ad->du;
        rate = st.ad_rate0 * exp(st.ad_slope * ((st.rk_stage == 0 ? u : u + dt) - st.ad_u0));
    }
    const double kR = (st.kappa ? st.kappa[b] : 1.0) * rate;
    bool bad = false;
    double errmax = 0.0;
#pragma unroll
    for (int q = 0; q < kMaxPerThread; ++q) {
        const int i = tid + q * KX_CTA;
        if (i >= N) continue;
        const size_t o = (size_t)b * N + i;
        double s = 0.0;
        for (int r = 0; r < st.nsrc; ++r) s += st.amp[r] * st.G[(size_t)r * N + i];
        const double k = kR * C[q] + s;
        const double f0 = st.f[o];
        double next;      // input of the next operator evaluation
        if (st.rk_method == KX_EULER) {
            next = f0 + dt * k;
            st.f[o] = next;
        } else if (st.rk_method == KX_HEUN) {
            if (st.rk_stage == 0) { st.k1[o] = k; next = f0 + dt * k; st.fstage[o] = next; }
            else { next = f0 + 0.5 * dt * (st.k1[o] + k); st.f[o] = next; }
        } else if (st.rk_method == KX_HEUN_ADAPT) {
            if (st.rk_stage == 0) { st.k1[o] = k; next = f0 + dt * k; st.fstage[o] = next; }      // Euler predictor
            else {                                                                                  // Heun corrector, kept aside
                next = f0 + 0.5 * dt * (st.k1[o] + k);
                st.k2[o] = next;
                const double e = fabs(next - st.fstage[o]) / (st.ad_atol + st.ad_rtol * fmax(fabs(f0), fabs(next)));
                errmax = isfinite(e) ? fmax(errmax, e) : INFINITY;
            }
        } else {
            if (st.rk_stage == 0) { st.k1[o] = k; next = f0 + 0.5 * dt * k; st.fstage[o] = next; }
            else if (st.rk_stage == 1) { st.k2[o] = k; next = f0 + 0.5 * dt * k; st.fstage[o] = next; }
            else if (st.rk_stage == 2) { st.k3[o] = k; next = f0 + dt * k; st.fstage[o] = next; }
            else { next = f0 + (dt / 6.0) * (st.k1[o] + 2.0 * st.k2[o] + 2.0 * st.k3[o] + k); st.f[o] = next; }
        }
        if (!isfinite(next)) bad = true;
        s_y[i] = kx_yval(next, d.interp, d.f_floor, d.eta);
    }
    if (bad && st.rk_method != KX_HEUN_ADAPT) atomicOr(st.flag, 1);      // a rejected attempt may overflow harmlessly
    if (st.rk_method == KX_HEUN_ADAPT && st.rk_stage == 1) {
        const double e = block_max(errmax, s_red);                         // order independent: deterministic
        if (tid == 0) atomicMax(&st.ad->errkey, kx_dkey(e));
    }
    __syncthreads();
    if (st.ydnext) {
        double2* ydn = reinterpret_cast<double2*>(st.ydnext) + (size_t)b * N;
        for (int i = tid; i < N; i += KX_CTA) {
            const double y0 = s_y[i], y1 = (i + 1 < N) ? s_y[i + 1] : y0;
            ydn[i] = make_double2(y0, y1 - y0);
        }
    }
}

// ---------------------------------------------------------------- adaptive Heun: accept / reject, controller update
// k_adapt_accept: one CTA per member; every CTA reads the same error norm and takes the same decision.
__global__ void __launch_bounds__(KX_CTA) k_adapt_accept(int N, double* __restrict__ f, const double* __restrict__ fnew,
                                                         const KxAdapt* __restrict__ ad, int* __restrict__ flag)
{
    if (ad->done) return;
    const long long k = ad->errkey;
    const double err = __longlong_as_double(k >= 0 ? k : (k ^ 0x7fffffffffffffffLL));
    if (!(err <= 1.0)) return;                                   // rejected (also when err is inf / nan)
    bool bad = false;
    for (int i = threadIdx.x; i < N; i += KX_CTA) {
        const double v = fnew[(size_t)blockIdx.x * N + i];
        f[(size_t)blockIdx.x * N + i] = v;
        if (!isfinite(v)) bad = true;
    }
    if (bad) atomicOr(flag, 1);
}

// k_adapt_ctrl: one thread.  du <- du clamp(safety / sqrt(err), 0.2, 5); accepted: u <- u + du_old, du <= u1 - u.
__global__ void k_adapt_ctrl(KxAdapt* ad, double u1, double safety)
{
    if (ad->done) return;
    const long long k = ad->errkey;
    const double err = __longlong_as_double(k >= 0 ? k : (k ^ 0x7fffffffffffffffLL));
    const bool ok = err <= 1.0;
    double fac = safety / sqrt(fmax(err, 1e-10));
    if (!(fac == fac)) fac = 0.2;                                // nan error: shrink
    fac = fmin(fmax(fac, 0.2), 5.0);
    double u = ad->u, du = ad->du;
    if (ok) { u += du; ad->accepted += 1; } else { ad->rejected += 1; }
    du *= fac;
    if (u1 - u <= 1e-14 * fmax(fabs(u1), 1.0)) { ad->done = 1; u = u1; }
    else if (du > u1 - u) du = u1 - u;
    ad->u = u; ad->du = du;
    ad->errkey = kx_dkey(0.0);
}

// ---------------------------------------------------------------- monoenergetic source deposition
__global__ void __launch_bounds__(KX_CTA) k_delta_source(KxDev d, double p0, double* __restrict__ G)
{
    __shared__ int s_L;
    const int N = d.N;
    if (threadIdx.x == 0) {            // largest L <= N-2 with p_L <= p0
        int lo = 0, hi = N - 2;
        while (lo < hi) {
            int mid = (lo + hi + 1) >> 1;
            if (d.p[mid] <= p0) lo = mid; else hi = mid - 1;
        }
        s_L = lo;
    }
    __syncthreads();
    const int L = s_L;
    const double E0 = sqrt(p0 * p0 + d.m * d.m);
    const double aR = (E0 - d.E[L]) / (d.E[L + 1] - d.E[L]);      // energy-linear deposition fractions
    for (int i = threadIdx.x; i < N; i += KX_CTA)
        G[i] = i == L ? (1.0 - aR) / d.h[L] : (i == L + 1 ? aR / d.h[L + 1] : 0.0);
}

// ---------------------------------------------------------------- a9: moments, eq. B.2
__global__ void __launch_bounds__(KX_CTA)
k_moments(KxDev d, const double* __restrict__ f, double* n, double* rho, double* p1, double* p2, int stride)
{
    __shared__ double s_red[8 * 8];
    const int N = d.N, b = blockIdx.x;
    double v[4] = {0.0, 0.0, 0.0, 0.0};
    for (int i = threadIdx.x; i < N; i += KX_CTA) {
        const double hf = d.h[i] * f[(size_t)b * N + i];
        const double p = d.p[i];
        v[0] += hf;
        v[1] += hf * d.E[i];
        v[2] += hf * p;
        v[3] += hf * p * p;
    }
    block_sum<4>(v, s_red);
    if (threadIdx.x == 0) {
        const double fac = d.g_chi / (2.0 * 3.14159265358979323846 * 3.14159265358979323846);
        if (n) n[(size_t)b * stride] = fac * v[0];
        if (rho) rho[(size_t)b * stride] = fac * v[1];
        if (p1) p1[(size_t)b * stride] = v[0] != 0.0 ? v[2] / v[0] : 0.0;
        if (p2) p2[(size_t)b * stride] = v[0] != 0.0 ? v[3] / v[0] : 0.0;
    }
}

template <int BT, int MODE, int QS>
cudaError_t launch_contract_t(const KxDev& d, int sm_count, const double* f, const double* yd,
                              double* part, int B, const long long* mstat, bool pdl, cudaStream_t s)
{
    const int N = d.N;
    size_t smem = (size_t)BT * N * 24 + (size_t)(KX_CTA / 32) * (QS ? 4 : 2) * BT * 8
                + (MODE == MODE_LOG_TAB ? (size_t)(KX_EXP_REP << KX_EXP_BITS) * 8 : 0) + (size_t)(N + 1) * 4;
    cudaError_t e = cudaFuncSetAttribute(k_contract<BT, MODE, QS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int occ = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_contract<BT, MODE, QS>, KX_CTA, smem);
    if (e != cudaSuccess) return e;
    if (occ < 1) occ = 1;
    const int groups = (B + BT - 1) / BT;
    int gx = (sm_count * occ + groups - 1) / groups;
    if (gx < 1) gx = 1;
    dim3 grid(gx, groups);
    return kx_launch(k_contract<BT, MODE, QS>, grid, dim3(KX_CTA), smem, s, pdl, d, f, reinterpret_cast<const double2*>(yd), part, B, mstat);
}

template <int BT>
cudaError_t launch_contract_m(const KxDev& d, int sm_count, const double* f, const double* yd,
                              double* part, int B, const long long* mstat, bool pdl, cudaStream_t s)
{
    if (d.eta) {         // quantum statistics: LOG interpolation only (checked in kx_build)
        if (d.exp_impl == KX_EXP_LIBM) return launch_contract_t<BT, MODE_LOG_LIBM, 1>(d, sm_count, f, yd, part, B, mstat, pdl, s);
        return launch_contract_t<BT, MODE_LOG_TAB, 1>(d, sm_count, f, yd, part, B, mstat, pdl, s);
    }
    if (d.interp == KX_INTERP_LINEAR) return launch_contract_t<BT, MODE_LINEAR, 0>(d, sm_count, f, yd, part, B, mstat, pdl, s);
    if (d.exp_impl == KX_EXP_LIBM) return launch_contract_t<BT, MODE_LOG_LIBM, 0>(d, sm_count, f, yd, part, B, mstat, pdl, s);
    return launch_contract_t<BT, MODE_LOG_TAB, 0>(d, sm_count, f, yd, part, B, mstat, pdl, s);
}

}  // namespace

int kx_pick_bt(int N, int B)
{
    int cap = N > 512 ? 4 : 8;
    int bt = 1;
    while (bt < B && bt < cap) bt <<= 1;
    return bt;
}

int kx_pick_chunk(long long nnz_est, int N, int B, int sm_count)
{
    const int bt = kx_pick_bt(N, B);
    const long long groups = (B + bt - 1) / bt;
    long long c = nnz_est * groups / ((long long)sm_count * 12);
    c = (c / KX_CTA) * KX_CTA;
    if (c < 1024) c = 1024;
    if (c > 8192) c = 8192;
    return (int)c;
}

cudaError_t kx_launch_prep(const KxDev& d, const double* f, double* yd, int B, cudaStream_t s)
{
    dim3 grid((d.N + 255) / 256, B);
    k_prep<<<grid, 256, 0, s>>>(d, f, reinterpret_cast<double2*>(yd), B);
    return cudaGetLastError();
}

cudaError_t kx_launch_contract(const KxDev& d, int sm_count, const double* f, const double* yd,
                               double* part, int B, const long long* mstat, bool pdl, cudaStream_t s)
{
    switch (kx_pick_bt(d.N, B)) {
        case 1: return launch_contract_m<1>(d, sm_count, f, yd, part, B, mstat, pdl, s);
        case 2: return launch_contract_m<2>(d, sm_count, f, yd, part, B, mstat, pdl, s);
        case 4: return launch_contract_m<4>(d, sm_count, f, yd, part, B, mstat, pdl, s);
        default: return launch_contract_m<8>(d, sm_count, f, yd, part, B, mstat, pdl, s);
    }
}

cudaError_t kx_launch_finish(const KxDev& d, const double* fin, const double* part, int B,
                             const KxStage& st, cudaStream_t s)
{
    if (st.gpart) {
        cudaError_t e = kx_launch(k_reduce, dim3(st.NT, (B + 1) / 2), dim3(256), 0, s, true, d.N, B, st);
        if (e != cudaSuccess) return e;
        if (st.fb_f) {
            e = kx_launch_contract(d, st.fb_sm_count, st.fb_f, st.fb_yd, st.fb_part, B, st.mstat, true, s);
            if (e != cudaSuccess) return e;
        }
    }
    return kx_launch(k_finish, dim3(B), dim3(KX_CTA), 0, s, true, d, fin, part, B, st);
}

cudaError_t kx_launch_adapt_step(const KxDev& d, double* f, const double* fnew, int B, KxAdapt* ad, double u1, double safety,
                                 int* flag, cudaStream_t s)
{
    k_adapt_accept<<<B, KX_CTA, 0, s>>>(d.N, f, fnew, ad, flag);
    k_adapt_ctrl<<<1, 1, 0, s>>>(ad, u1, safety);
    return cudaGetLastError();
}

cudaError_t kx_launch_delta_source(const KxDev& d, double p0, double* G, cudaStream_t s)
{
    k_delta_source<<<1, KX_CTA, 0, s>>>(d, p0, G);
    return cudaGetLastError();
}

cudaError_t kx_launch_moments(const KxDev& d, const double* f, int B, double* n, double* rho,
                              double* p1, double* p2, int stride, cudaStream_t s)
{
    k_moments<<<B, KX_CTA, 0, s>>>(d, f, n, rho, p1, p2, stride);
    return cudaGetLastError();
}
