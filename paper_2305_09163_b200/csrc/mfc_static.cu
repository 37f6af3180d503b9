// mfc_cfl_dt_static (include/mfc.h): the CFL time step for callers that must not allocate device memory.
//
// Who that is.  mfc_init reserves the library's workspace with cudaMalloc, and so does every entry point that takes a
// context.  Some hosts cannot let a library do that:
//   * a solver embedded in an application whose own pool already holds the whole device (a framework's caching allocator
//     run with its memory fraction at 1, a job scheduler that caps the process' device memory at what the application
//     reserved): a further cudaMalloc fails there, or takes memory the application counted on;
//   * a time loop with other streams in flight: cudaMalloc and cudaFree synchronise the whole device, so a library that
//     allocates (even once, lazily, at an unpredictable call) stalls every other stream of the process;
//   * plug-in code that is handed device buffers and a stream and is told to enqueue work on them and nothing else.
// This entry point serves them: it takes the grid and the equation of state as plain arguments (no context), the state
// and the result as device pointers of the caller, and keeps the one piece of workspace the reduction needs -- one
// partial maximum per block and a ticket counter -- in a fixed array that is part of the library's image.
//
// What it costs.  The array below is MFC_STATIC_SCRATCH_BYTES (about 64 KiB) of device memory on EVERY device that loads
// libmfc_b200, from the load until the process exits, used or not.  Its size fixes the largest grid the entry point takes
// (MFC_STATIC_MAX_CELLS interior cells); larger grids are refused with MFC_ELIMIT, nothing is truncated.
//
// What the caller has to know.
//   * The first call on a device asks the runtime for the device address of the array (cudaGetSymbolAddress) and keeps
//     it; make that first call outside any stream capture.  No call allocates: there is no cudaMalloc, cudaFree,
//     cudaMallocHost or library routine that allocates anywhere in this file.
//   * All calls on a device share the array, and it keeps what the previous call left in it.  Every call therefore
//     clears the ticket counter on the caller's stream before its kernel; the partial maxima need no clearing (every
//     block of a launch writes its slot before any slot is read).  Two calls whose kernels can overlap on the GPU
//     (different streams, no dependency between them) would count each other's tickets and mix partial maxima: the
//     results of both are then undefined.  Order such calls (one stream, or an event between the two).
//   * Uniform grids only (the tables of a non-uniform grid are workspace of a size this array is not meant for).
//
// The arithmetic is the context path's (cell_signal_speed of mfc_kernels.cuh), the reduction is a maximum
// of bit patterns (exact in any order), and dt = cfl * (1 / max) is formed with IEEE division and multiplication as
// mfc_cfl_dt forms it on the host: the two entry points return the same bits.
#include "../../include/mfc.h"
#include "mfc_kernels.cuh"

#include <cmath>
#include <cstring>
#include <mutex>

namespace mfc {

constexpr int STATIC_THREADS = 256;
constexpr int STATIC_TRIPS = MFC_STATIC_CELLS_PER_BLOCK / STATIC_THREADS;   // cells of one thread
constexpr int STATIC_HEAD = 32;   // slot 0: ticket counter; the partial maxima start 256 bytes in
static_assert(MFC_STATIC_CELLS_PER_BLOCK % (2 * STATIC_THREADS) == 0, "two cells per thread and trip");
static_assert(sizeof(unsigned long long) * (STATIC_HEAD + MFC_STATIC_MAX_BLOCKS) == MFC_STATIC_SCRATCH_BYTES, "mfc.h states the size");

// The workspace.  In HOST code this name is only a handle for cudaGetSymbolAddress / cudaMemcpyToSymbol: it is not a
// device address, and a kernel given `cfl_static_scratch` from the host would read and write whatever host memory the
// handle happens to be (or fault).  static_scratch() below turns it into the device address, once per device.
static __device__ __align__(256) unsigned long long cfl_static_scratch[STATIC_HEAD + MFC_STATIC_MAX_BLOCKS];

// Block b owns the interior cells [b * CELLS_PER_BLOCK, (b + 1) * CELLS_PER_BLOCK) (x fastest) and leaves their maximum
// signal speed over dx in scratch[HEAD + b]; the block that draws the last ticket reduces the partial maxima and writes
// dt.  The maximum is taken on bit patterns exactly as in cfl_kernel: NaN and +inf order above every finite speed, so an
// inadmissible cell makes dt NaN (or 0) instead of being dropped.
template <int D, int NF>
__global__ void __launch_bounds__(STATIC_THREADS) cfl_static_kernel(Geo g, Eos eos_in, double cfl, const double *__restrict__ q,
                                                                    unsigned long long *scratch, double *dt_out)
{
    using I = Idx<D, NF>;
    // reciprocal seeds of gamma_i - 1 (mfc_init computes them with a kernel of its own and a temporary buffer; here every
    // thread derives them: 3 x 6 FP64 instructions)
    Eos eos = eos_in;
#pragma unroll
    for (int i = 0; i < NF; ++i) eos.ygm1[i] = div_seed(eos.gm1[i]);
    const unsigned ncell = (unsigned)g.n[0] * (unsigned)g.n[1] * (unsigned)g.n[2];   // <= MFC_STATIC_MAX_CELLS < 2^32
    const unsigned n0 = (unsigned)g.n[0], n1 = (unsigned)g.n[1];
    const double inv[3] = {g.inv_dx[0], g.inv_dx[1], g.inv_dx[2]};
    auto cell_of = [&](unsigned f) -> long long {
        const unsigned r = f / n0;
        const int i = (int)(f - r * n0);
        const int k = (int)(r / n1), j = (int)(r - (unsigned)k * n1);
        return (long long)(k + g.g[2]) * g.sz + (long long)(j + g.g[1]) * g.sy + (i + g.g[0]);
    };
    auto bits = [](double s) -> unsigned long long {
        return (unsigned long long)__double_as_longlong(s == s ? s : __longlong_as_double(0x7ff8000000000000ll));
    };
    unsigned long long best = 0ull;
    const unsigned first = blockIdx.x * (unsigned)MFC_STATIC_CELLS_PER_BLOCK + threadIdx.x;
    for (int t = 0; t < STATIC_TRIPS; t += 2) {
        const unsigned f0 = first + (unsigned)t * STATIC_THREADS, f1 = f0 + STATIC_THREADS;
        if (f0 >= ncell) break;
        const long long c0 = cell_of(f0), c1 = cell_of(f1 < ncell ? f1 : f0);
        double q0[I::NEQ], q1[I::NEQ];
#pragma unroll
        for (int e = 0; e < I::NEQ; ++e) { q0[e] = __ldg(q + (long long)e * g.cells + c0); q1[e] = __ldg(q + (long long)e * g.cells + c1); }
        const unsigned long long b0 = bits(cell_signal_speed<D, NF>(inv, eos, q0)), b1 = bits(cell_signal_speed<D, NF>(inv, eos, q1));
        best = max(best, max(b0, b1));
    }
    __shared__ unsigned long long red[STATIC_THREADS / 32];
    __shared__ bool last;
    auto block_max = [&](unsigned long long v) -> unsigned long long {   // valid in thread 0
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) v = max(v, __shfl_xor_sync(0xffffffffu, v, off));
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
        __syncthreads();
        if (threadIdx.x == 0)
            for (int w = 1; w < STATIC_THREADS / 32; ++w) v = max(v, red[w]);
        return v;
    };
    best = block_max(best);
    if (threadIdx.x == 0) {
        scratch[STATIC_HEAD + blockIdx.x] = best;
        __threadfence();                                                 // the partial maximum before the ticket
        last = atomicAdd(scratch, 1ull) == (unsigned long long)gridDim.x - 1ull;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();                                                     // the other blocks' slots after the last ticket
    unsigned long long all = 0ull;
    for (unsigned b = threadIdx.x; b < gridDim.x; b += STATIC_THREADS) all = max(all, __ldcg(scratch + STATIC_HEAD + b));
    __syncthreads();                                                     // red[] is reused
    all = block_max(all);
    if (threadIdx.x == 0) {
        const double v = __longlong_as_double((long long)all);
        *dt_out = __dmul_rn(cfl, __ddiv_rn(1.0, v));                     // mfc_cfl_dt: cfl * (1.0 / v) on the host
        scratch[0] = 0ull;                                               // leaves the counter as the next call needs it
    }
}

namespace {

constexpr int MAX_DEVICES = 64;
std::mutex static_mutex;
unsigned long long *static_ptr[MAX_DEVICES] = {};    // device address of cfl_static_scratch per device ordinal

// device address of the workspace on `dev`, which must be the CURRENT device: a __device__ array exists once per
// device, and cudaGetSymbolAddress answers for the device that is current when it is called
cudaError_t static_scratch(int dev, unsigned long long **out)
{
    std::lock_guard<std::mutex> lock(static_mutex);
    if (!static_ptr[dev]) {
        unsigned long long *p = nullptr;
        const cudaError_t err = cudaGetSymbolAddress((void **)&p, cfl_static_scratch);
        if (err != cudaSuccess) return err;
        static_ptr[dev] = p;
    }
    *out = static_ptr[dev];
    return cudaSuccess;
}

template <int D>
cudaError_t launch_static(int nf, unsigned blocks, const Geo &g, const Eos &e, double cfl, const double *q,
                          unsigned long long *scratch, double *dt, cudaStream_t s)
{
    switch (nf) {
        case 1: cfl_static_kernel<D, 1><<<blocks, STATIC_THREADS, 0, s>>>(g, e, cfl, q, scratch, dt); break;
        case 2: cfl_static_kernel<D, 2><<<blocks, STATIC_THREADS, 0, s>>>(g, e, cfl, q, scratch, dt); break;
        case 3: cfl_static_kernel<D, 3><<<blocks, STATIC_THREADS, 0, s>>>(g, e, cfl, q, scratch, dt); break;
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

}  // namespace
}  // namespace mfc

extern "C" int mfc_cfl_dt_static(const mfc_grid *grid, int n_fluids, const mfc_fluid *eos, double cfl, int device,
                                 const double *q_dev, double *dt_dev, void *stream)
{
    using namespace mfc;
    // ---- arguments: everything that can be refused is refused before the first CUDA call ----
    if (!grid || !eos || !q_dev || !dt_dev) return MFC_EINVAL;
    if (grid->ndim < 1 || grid->ndim > 3 || n_fluids < 1) return MFC_EINVAL;
    if (n_fluids > MFC_MAX_FLUIDS) return MFC_EUNSUPPORTED;
    long long ncell = 1;
    for (int d = 0; d < grid->ndim; ++d) {
        if (grid->n[d] < MFC_NG) return MFC_EINVAL;
        if (grid->edges_host[d]) return MFC_EUNSUPPORTED;                // non-uniform spacing needs tables: use a context
        if (!(grid->hi[d] > grid->lo[d]) || !std::isfinite(grid->hi[d] - grid->lo[d])) return MFC_EINVAL;
        if (grid->inv_dx[d] != 0.0 && (!(grid->inv_dx[d] > 0.0) || !std::isfinite(grid->inv_dx[d]))) return MFC_EINVAL;
        ncell *= grid->n[d];
        if (ncell > MFC_STATIC_MAX_CELLS) return MFC_ELIMIT;             // (checked per factor: no overflow)
    }
    for (int i = 0; i < n_fluids; ++i)
        if (!(eos[i].gamma > 1.0) || !std::isfinite(eos[i].gamma) || !std::isfinite(eos[i].pi_inf)) return MFC_EINVAL;
    if (!(cfl > 0.0)) cfl = 0.3;                                         // as mfc_opts.cfl

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return MFC_ECUDA;
    if (device < 0 && cudaGetDevice(&device) != cudaSuccess) return MFC_ECUDA;
    if (device >= ndev) return MFC_EINVAL;
    if (device >= MAX_DEVICES) return MFC_EUNSUPPORTED;

    // ---- the launch description mfc_init would build (same expressions: same bits of 1 / dx) ----
    Geo g;
    std::memset(&g, 0, sizeof(g));
    g.ndim = grid->ndim;
    for (int d = 0; d < 3; ++d) {
        const bool act = d < grid->ndim;
        g.n[d] = act ? grid->n[d] : 1;
        g.g[d] = act ? NG : 0;
        g.p[d] = g.n[d] + 2 * g.g[d];
        g.inv_dx[d] = act ? (grid->inv_dx[d] > 0.0 ? grid->inv_dx[d] : (double)grid->n[d] / (grid->hi[d] - grid->lo[d])) : 1.0;
        g.bc_lo[d] = g.bc_hi[d] = MFC_BC_EXTRAP;                         // unused: the reduction reads interior cells only
    }
    g.sy = g.p[0];
    g.sz = (long long)g.p[0] * g.p[1];
    g.cells = g.sz * g.p[2];
    Eos e;
    std::memset(&e, 0, sizeof(e));
    double Gm[MAX_NF], Pm[MAX_NF];
    for (int i = 0; i < n_fluids; ++i) {
        e.gamma[i] = eos[i].gamma;
        e.pi_inf[i] = eos[i].pi_inf;
        e.gm1[i] = eos[i].gamma - 1.0;
        Gm[i] = 1.0 / (eos[i].gamma - 1.0);
        Pm[i] = eos[i].gamma * eos[i].pi_inf / (eos[i].gamma - 1.0);
    }
    e.G_last = Gm[n_fluids - 1];
    e.P_last = Pm[n_fluids - 1];
    for (int i = 0; i < n_fluids - 1; ++i) {
        e.dG[i] = Gm[i] - e.G_last;
        e.dP[i] = Pm[i] - e.P_last;
    }

    // ---- set-up (first call on this device) and launch, with the device current ----
    int prev = -1;
    if (cudaGetDevice(&prev) != cudaSuccess) return MFC_ECUDA;
    if (prev != device && cudaSetDevice(device) != cudaSuccess) return MFC_ECUDA;
    cudaStream_t s = (cudaStream_t)stream;
    unsigned long long *scratch = nullptr;
    cudaError_t err = static_scratch(device, &scratch);
    // the counter must start at zero whatever an earlier call (perhaps one that failed half way) left behind
    if (err == cudaSuccess) err = cudaMemsetAsync(scratch, 0, sizeof(unsigned long long), s);
    if (err == cudaSuccess) {
        const unsigned blocks = (unsigned)((ncell + MFC_STATIC_CELLS_PER_BLOCK - 1) / MFC_STATIC_CELLS_PER_BLOCK);
        switch (grid->ndim) {
            case 1: err = launch_static<1>(n_fluids, blocks, g, e, cfl, q_dev, scratch, dt_dev, s); break;
            case 2: err = launch_static<2>(n_fluids, blocks, g, e, cfl, q_dev, scratch, dt_dev, s); break;
            case 3: err = launch_static<3>(n_fluids, blocks, g, e, cfl, q_dev, scratch, dt_dev, s); break;
        }
    }
    if (prev != device) cudaSetDevice(prev);
    if (err != cudaSuccess) {
        cudaGetLastError();
        return MFC_ECUDA;
    }
    return MFC_OK;
}
