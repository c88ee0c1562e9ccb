// kx_static.cu -- kx_collide_static: one operator evaluation that ALLOCATES NOTHING.
//
// Some callers cannot call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid it.  Every
// other evaluation entry point of libkx may grow the handle's workspace on its first call with a larger batch.  This one
// is a variant of the fused streaming kernel k_stream (kx_stream.cuh: exact contraction a4-a5 -> grid barrier -> finishing
// phase a6-a7) whose scratch memory -- the per-task partial sums, the task table and the grid-barrier words -- lives in a
// file-scope `static __device__` array of fixed size (about 2 MiB; every GPU that loads the library holds it until exit).
// The caller passes inputs and outputs; the kernel tensor is the handle's own row storage (built by kx_build).
//
// In host code the array's NAME is a host-side stand-in, not a device address: its device address is taken once per device,
// with that device current, by cudaGetSymbolAddress (static_scratch() below) and handed to the kernels as a pointer.
//
// All calls share the array, which keeps the last call's contents: the barrier's arrival counter is cleared by the set-up
// kernel of every call, the task table is rewritten by it, and every partial that is read was written by the same call.
// Calls that overlap on one GPU (different streams, several host threads) RACE on the array: serialise them.
//
// Compiled with --fmad=false; fused multiply-adds are explicit.
#include "kx_device.cuh"

#include <atomic>
#include <mutex>

#define KX_STATIC_MAX_PAIRS 131072          // (task, member) pairs of partial sums the scratch holds: 2 MiB
#define KX_STATIC_BT        4               // members per contraction group
#define KX_STATIC_MAX_DEV   64

namespace {

using namespace kxd;

constexpr size_t kBarDoubles = 32;                                   // 256 bytes: barrier words (4 x uint32 used)
constexpr size_t kTaskDoubles = ((KX_MAX_N + 1) * 4 + 63) / 64 * 8;   // task table [N + 1] uint32, padded to 64 bytes
constexpr size_t kScratchDoubles = kBarDoubles + kTaskDoubles + (size_t)KX_STATIC_MAX_PAIRS * 2;

static __device__ __align__(256) double kx_static_scratch[kScratchDoubles];

// set-up kernel of every call (one CTA of 1024 threads): clears the barrier's arrival counter and writes the task table
// taskptr[i] = exclusive scan of ceil(len_i / chunk) for the chunk size of this call (N <= 1024)
__global__ void __launch_bounds__(1024) k_static_setup(KxDev d, int chunk, double* scratch)
{
    __shared__ unsigned s_warp[32];
    unsigned* bar = reinterpret_cast<unsigned*>(scratch);
    unsigned* taskptr = reinterpret_cast<unsigned*>(scratch + kBarDoubles);
    const int t = threadIdx.x;
    if (t == 0) bar[0] = 0u;
    unsigned cnt = 0;
    if (t < d.N) {
        const unsigned len = d.rowptr[t + 1] - d.rowptr[t];
        cnt = (len + (unsigned)chunk - 1u) / (unsigned)chunk;
    }
    unsigned v = cnt;
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned u = __shfl_up_sync(0xffffffffu, v, o);
        if ((t & 31) >= o) v += u;
    }
    if ((t & 31) == 31) s_warp[t >> 5] = v;
    __syncthreads();
    if (t < 32) {
        unsigned w = s_warp[t];
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned u = __shfl_up_sync(0xffffffffu, w, o);
            if (t >= o) w += u;
        }
        s_warp[t] = w;
    }
    __syncthreads();
    const unsigned excl = v - cnt + ((t >> 5) ? s_warp[(t >> 5) - 1] : 0u);
    if (t < d.N) taskptr[t] = excl;
    if (t == d.N - 1) taskptr[d.N] = excl + cnt;
}

// the variant of k_stream: `d.taskptr`, `st.part` and `st.bar` point into the static scratch
template <int MODE>
__global__ void __launch_bounds__(KX_CTA, 2)
k_collide_static(KxDev d, const double* __restrict__ f, int B, KxStage st)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double s_red[8 * 8];
    constexpr int BT = KX_STATIC_BT;
    const int groups = (B + BT - 1) / BT;
    for (int g = blockIdx.y; g < groups; g += gridDim.y)
        contract_group<BT, MODE, 0>(d, f, nullptr, st.part, B, g * BT, blockIdx.x, gridDim.x, smem_raw);
    grid_barrier(st.bar, st.epoch);
    const unsigned cta = blockIdx.y * gridDim.x + blockIdx.x, nctas = gridDim.x * gridDim.y;
    double* scr = reinterpret_cast<double*>(smem_raw);
    for (int b = (int)cta; b < B; b += (int)nctas) {
        if (d.N <= KX_CTA) finish_member<1>(d, f, B, st, nullptr, false, b, scr, s_red, nullptr);
        else if (d.N <= 2 * KX_CTA) finish_member<2>(d, f, B, st, nullptr, false, b, scr, s_red, nullptr);
        else finish_member<4>(d, f, B, st, nullptr, false, b, scr, s_red, nullptr);
    }
}

// ---------------------------------------------------------------- host side
std::mutex g_mu;
double* g_scratch[KX_STATIC_MAX_DEV];            // device address of kx_static_scratch on every device (null: not taken yet)
bool g_attr_done[KX_STATIC_MAX_DEV][3];
struct Occ { int N, occ; };
Occ g_occ[KX_STATIC_MAX_DEV][3];
std::atomic<unsigned> g_epoch{0};

// once per device, with that device current: the device address of the scratch array
cudaError_t static_scratch(int device, double** out)
{
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch[device]) {
        void* ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&ptr, kx_static_scratch);
        if (e != cudaSuccess) return e;
        g_scratch[device] = static_cast<double*>(ptr);
    }
    *out = g_scratch[device];
    return cudaSuccess;
}

template <int MODE>
cudaError_t launch_static(int device, int slot, const KxDev& d, int sm_count, const double* f, int B, KxStage& st, cudaStream_t s)
{
    const int N = d.N;
    size_t smem = contract_smem<KX_STATIC_BT, MODE, 0>(N);
    const size_t fin = finish_scratch_bytes(N, 0, 0, 0, 0);
    if (smem < fin) smem = fin;
    cudaError_t e;
    {
        std::lock_guard<std::mutex> lock(g_mu);
        if (!g_attr_done[device][slot]) {
            e = cudaFuncSetAttribute(k_collide_static<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, 226 * 1024);
            if (e != cudaSuccess) return e;
            g_attr_done[device][slot] = true;
        }
        if (g_occ[device][slot].N != N) {
            int occ = 0;
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_collide_static<MODE>, KX_CTA, smem);
            if (e != cudaSuccess) return e;
            g_occ[device][slot] = {N, occ < 1 ? 1 : occ};
        }
    }
    // every CTA must be resident (grid barrier): at most occ per SM; never more CTAs per member group than tasks
    const int cap = sm_count * g_occ[device][slot].occ;
    const int groups = (B + KX_STATIC_BT - 1) / KX_STATIC_BT;
    const int gy = groups < cap ? groups : cap;
    int gx = cap / gy;
    const long long tasks_bound = (long long)N + (long long)N * ((long long)N * (N + 1) / 2) / d.chunk;
    if ((long long)gx > tasks_bound) gx = (int)tasks_bound;
    if (gx < 1) gx = 1;
    return kx_launch_coop(k_collide_static<MODE>, dim3(gx, gy), dim3(KX_CTA), smem, s, d, f, B, st);
}

}  // namespace

extern "C" kx_status_t kx_collide_static(kx_handle_t h, const double* f, double* C, int32_t B, uint32_t flags, void* stream)
{
    if (!h) return KX_ERR_INVALID_ARG;
    if (!f || !C || B < 1) { h->err = "kx_collide_static: f or C is NULL, or B < 1"; return KX_ERR_INVALID_ARG; }
    if ((((uintptr_t)f | (uintptr_t)C) & 15u) != 0) { h->err = "kx_collide_static: device pointer not 16-byte aligned"; return KX_ERR_INVALID_ARG; }
    if (C == f) { h->err = "kx_collide_static: in place (C == f) is not allowed"; return KX_ERR_INVALID_ARG; }
    if (h->d.eta != 0 || h->d.prec != KX_FP64) {
        h->err = "kx_collide_static: classical statistics in fp64 only";
        return KX_ERR_UNSUPPORTED;
    }
    if (h->device < 0 || h->device >= KX_STATIC_MAX_DEV) { h->err = "kx_collide_static: device ordinal out of range"; return KX_ERR_UNSUPPORTED; }
    if (h->d.m_dev) { h->err = "kx_collide_static: the handle is inside kx_evolve_adaptive"; return KX_ERR_INVALID_ARG; }
    const int N = h->d.N;
    // entries per task: 4096, doubled until the (task, member) pairs fit the static scratch.  The number of stored entries
    // is known on the host unless the mass was changed since (then every triple is assumed kept).
    const long long nnz_bound = h->nnz_stale ? (long long)N * ((long long)N * (N + 1) / 2) : h->nnz;
    int chunk = 4096;
    while (chunk < 65536 && (nnz_bound / chunk + N) * (long long)B > KX_STATIC_MAX_PAIRS) chunk *= 2;
    if ((nnz_bound / chunk + N) * (long long)B > KX_STATIC_MAX_PAIRS) {
        char buf[256];
        snprintf(buf, sizeof buf, "kx_collide_static: (tasks x members) = %lld x %d exceeds the static scratch of %d pairs "
                 "(2 MiB); use kx_collide or a smaller batch", nnz_bound / chunk + N, (int)B, KX_STATIC_MAX_PAIRS);
        h->err = buf;
        return KX_ERR_UNSUPPORTED;
    }
    int prev = -1;
    if (cudaGetDevice(&prev) != cudaSuccess) { h->err = "kx_collide_static: cudaGetDevice failed"; return KX_ERR_CUDA; }
    if (prev != h->device && cudaSetDevice(h->device) != cudaSuccess) { h->err = "kx_collide_static: cudaSetDevice failed"; return KX_ERR_CUDA; }
    kx_status_t rc = KX_OK;
    cudaStream_t s = (cudaStream_t)stream;
    double* scratch = nullptr;
    cudaError_t e = static_scratch(h->device, &scratch);
    if (e == cudaSuccess) {
        KxDev d = h->d;                                            // a copy: the handle's own task table is not touched
        d.chunk = chunk;
        d.taskptr = reinterpret_cast<unsigned*>(scratch + kBarDoubles);
        k_static_setup<<<1, 1024, 0, s>>>(d, chunk, scratch);
        e = cudaGetLastError();
        if (e == cudaSuccess) {
            KxStage st = {};
            st.flags = flags & KX_PROJECT;
            st.C = C; st.diag_stride = 4; st.evolve = 0;
            st.part = scratch + kBarDoubles + kTaskDoubles;
            st.bar = reinterpret_cast<unsigned*>(scratch);
            st.epoch = ++g_epoch;                                  // never the value a previous call left in bar[1]
            if (st.epoch == 0u) st.epoch = ++g_epoch;
            if (d.interp == KX_INTERP_LINEAR) e = launch_static<MODE_LINEAR>(h->device, 2, d, h->sm_count, f, B, st, s);
            else if (d.exp_impl == KX_EXP_LIBM) e = launch_static<MODE_LOG_LIBM>(h->device, 1, d, h->sm_count, f, B, st, s);
            else e = launch_static<MODE_LOG_TAB>(h->device, 0, d, h->sm_count, f, B, st, s);
        }
    }
    if (e != cudaSuccess) {
        h->err = std::string("kx_collide_static: ") + cudaGetErrorString(e);
        rc = KX_ERR_CUDA;
    }
    if (prev != h->device) cudaSetDevice(prev);
    return rc;
}
