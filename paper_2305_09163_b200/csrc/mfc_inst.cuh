// Launchers of every kernel family for one value of D (= MFC_D, set by the including translation unit), all
// NF in {1,2,3}.  One translation unit per D keeps the sm_100a compile parallel.
#include "mfc_kernels.cuh"

#ifndef MFC_D
#error "define MFC_D (1, 2 or 3) before including mfc_inst.cuh"
#endif
#define MFC_CAT2(a, b) a##b
#define MFC_CAT(a, b) MFC_CAT2(a, b)

namespace mfc {

#define MFC_FOR_NF(nf, STMT)                                                                                          \
    switch (nf) {                                                                                                     \
        case 1: { constexpr int NF = 1; STMT; } break;                                                                \
        case 2: { constexpr int NF = 2; STMT; } break;                                                                \
        case 3: { constexpr int NF = 3; STMT; } break;                                                                \
        default: return cudaErrorInvalidValue;                                                                        \
    }

cudaError_t MFC_CAT(launch_prim_d, MFC_D)(int nf, const Geo &g, const Eos &e, const double *q, double *w, cudaStream_t s)
{
    constexpr int D = MFC_D;
    const unsigned blocks = (unsigned)((g.cells + 255) / 256);
    MFC_FOR_NF(nf, (prim_kernel<D, NF><<<blocks, 256, 0, s>>>(g, e, q, w)))
    return cudaGetLastError();
}

template <int D, int NF>
static void launch_x(const Geo &g, const Eos &e, const double *w, const SweepOut &o, cudaStream_t s)
{
    constexpr int NEQ = 2 * NF + D;
    constexpr int bytes = sweep_x_smem_bytes<NEQ>();
    const long long G = (long long)g.n[1] * g.n[2] * g.p[0];
    const long long ntiles = (G - 2 * NG + (XT - 2) - 1) / (XT - 2);
    const long long cap = 2LL * (g.sms > 0 ? g.sms : 148);            // two resident blocks per multiprocessor
    const unsigned blocks = (unsigned)(ntiles < cap ? ntiles : cap);
    cudaFuncSetAttribute(sweep_x_kernel<D, NF>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    sweep_x_kernel<D, NF><<<blocks, XT, bytes, s>>>(g, e, w, o, (int)ntiles);
}

template <int D, int NF, int DIR>
static void launch_march(const Geo &g, const Eos &e, const double *w, const SweepOut &o, int segment, cudaStream_t s)
{
    constexpr int OTH = DIR == 1 ? 2 : 1;
    constexpr int NEQ = 2 * NF + D;
    constexpr int bytes = sweep_march_smem_bytes<NEQ>();
    const int nm = g.n[DIR];
    const int seg = segment < 1 ? 1 : (segment > nm ? nm : segment);
    const int nseg = (nm + seg - 1) / seg;
    const long long threads = (long long)g.n[0] * g.n[OTH] * nseg;
    const unsigned blocks = (unsigned)((threads + MBT - 1) / MBT);
    cudaFuncSetAttribute(sweep_march_kernel<D, NF, DIR>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    cudaFuncSetAttribute(sweep_march_kernel<D, NF, DIR>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    sweep_march_kernel<D, NF, DIR><<<blocks, MBT, bytes, s>>>(g, e, w, o, seg, nseg);
}

cudaError_t MFC_CAT(launch_sweep_d, MFC_D)(int nf, int dir, const Geo &g, const Eos &e, const double *w, const SweepOut &o,
                                           int segment, cudaStream_t s)
{
    constexpr int D = MFC_D;
    if (dir < 0 || dir >= D) return cudaErrorInvalidValue;
    if (dir == 0) {
        MFC_FOR_NF(nf, (launch_x<D, NF>(g, e, w, o, s)))
    }
#if MFC_D >= 2
    else if (dir == 1) {
        MFC_FOR_NF(nf, (launch_march<D, NF, 1>(g, e, w, o, segment, s)))
    }
#endif
#if MFC_D >= 3
    else if (dir == 2) {
        MFC_FOR_NF(nf, (launch_march<D, NF, 2>(g, e, w, o, segment, s)))
    }
#endif
    return cudaGetLastError();
}

cudaError_t MFC_CAT(launch_cfl_d, MFC_D)(int nf, const Geo &g, const Eos &e, const double *q, unsigned long long *min_bits,
                                         cudaStream_t s)
{
    constexpr int D = MFC_D;
    const long long ncell = (long long)g.n[0] * g.n[1] * g.n[2];
    long long want = (ncell + 255) / 256;
    const unsigned blocks = (unsigned)(want < 148 * 8 ? (want < 1 ? 1 : want) : 148 * 8);
    MFC_FOR_NF(nf, (cfl_kernel<D, NF><<<blocks, 256, 0, s>>>(g, e, q, min_bits)))
    return cudaGetLastError();
}

template <int D, int NF, int DIR>
static void launch_line_t(const Eos &e, int n, const double *w, double *vL, double *vR, double *F, double *uf, cudaStream_t s)
{
    line_weno_kernel<D, NF, DIR><<<(n + 2 + 127) / 128, 128, 0, s>>>(e, n, w, vL, vR);
    line_hllc_kernel<D, NF, DIR><<<(n + 1 + 127) / 128, 128, 0, s>>>(e, n, vL, vR, F, uf);
}

cudaError_t MFC_CAT(launch_line_d, MFC_D)(int nf, int dir, const Eos &e, int n, const double *w, double *vL, double *vR,
                                          double *F, double *uf, cudaStream_t s)
{
    constexpr int D = MFC_D;
    if (dir < 0 || dir >= D) return cudaErrorInvalidValue;
    if (dir == 0) { MFC_FOR_NF(nf, (launch_line_t<D, NF, 0>(e, n, w, vL, vR, F, uf, s))) }
#if MFC_D >= 2
    else if (dir == 1) { MFC_FOR_NF(nf, (launch_line_t<D, NF, 1>(e, n, w, vL, vR, F, uf, s))) }
#endif
#if MFC_D >= 3
    else if (dir == 2) { MFC_FOR_NF(nf, (launch_line_t<D, NF, 2>(e, n, w, vL, vR, F, uf, s))) }
#endif
    return cudaGetLastError();
}

}  // namespace mfc
