// Launchers of every kernel family for one value of D (= MFC_D, set by the including translation unit), all
// NF in {1,2,3}.  One translation unit per D keeps the sm_100a compile parallel.
#include <atomic>
#include "mfc_kernels.cuh"
#include "mfc_fused.cuh"
#include "mfc_fused_tma.cuh"
#include "mfc_fused_roles.cuh"

#ifndef MFC_D
#error "define MFC_D (1, 2 or 3) before including mfc_inst.cuh"
#endif
// rows of the 3D tile (a multiple of 4: whole warps per scheduler); -DMFC_TY_2F=8 / 16 build the variants measured in
// DESIGN.md 6.1
#ifndef MFC_TY_2F
#define MFC_TY_2F 12
#endif
// rows of the tile of the kernel with specialised Z warps (mfc_fused_roles.cuh)
#ifndef MFC_ROLES_TY
#define MFC_ROLES_TY 12
#endif
#define MFC_CAT2(a, b) a##b
#define MFC_CAT(a, b) MFC_CAT2(a, b)

namespace mfc {

#define MFC_FOR_ORDER(order, STMT)                                                                                    \
    switch (order) {                                                                                                  \
        case 1: { constexpr int ORDER = 1; STMT; } break;                                                             \
        case 3: { constexpr int ORDER = 3; STMT; } break;                                                             \
        case 5: { constexpr int ORDER = 5; STMT; } break;                                                             \
        default: return cudaErrorInvalidValue;                                                                        \
    }

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

// tile height of the fused kernel: 3D tiles of 12 rows (12 warps, 168 registers per thread); the staged plane, the
// exchange and staging buffers take 130 - 215 KB of shared memory, the z window of every column lives in TMEM
template <int D, int NF>
constexpr int fused_ty()
{
    if (D == 1) return 1;
    if (D == 2) return 8;
    return MFC_TY_2F;
}

// z segment of the march: blocks = tiles * nseg should fill whole waves of the multiprocessors (one block per
// multiprocessor), and every segment pays for 6 extra planes of load + cons->prim + z reconstruction: `fill` full planes
// of work (about 2 in the one-loop kernels; about 1 in the kernel with Z warps, measured: 128^3 is 1.6 % faster with
// 10 segments of 13 planes than with 3 of 43)
static int fused_segment(const Geo &g, long long tiles, int wanted, double fill = 2.0)
{
    const int nz = g.n[2];
    if (wanted > 0) return wanted < nz ? wanted : nz;
    const long long sms = g.sms > 0 ? g.sms : 148;
    double best = 1e300;
    int best_seg = nz;
    for (int nseg = 1; nseg <= (nz + 3) / 4; ++nseg) {
        const int seg = (nz + nseg - 1) / nseg;
        const long long blocks = tiles * ((nz + seg - 1) / seg);
        const double cost = (double)((blocks + sms - 1) / sms) * (seg + fill);
        if (cost < best) { best = cost; best_seg = seg; }
    }
    return best_seg;
}

// The opt-in to more than 48 KB of dynamic shared memory is a property of the kernel ON ONE DEVICE (the function handle
// belongs to the primary context of the device that is current): set once per instantiation and device (a function-local
// table of launch_fused<D, NF, ORDER>, indexed by the current device; mfc_opts.device allows contexts on several GPUs in
// one process), and its status kept: a failed opt-in is reported by every later launch on that device.  Device ordinals
// past the table set the attribute on every launch (microseconds).
constexpr int MFC_OPTIN_DEVICES = 64;
#define MFC_OPTIN_SHARED(kernel, bytes)                                                                               \
    [&]() -> cudaError_t {                                                                                            \
        static std::atomic<int> st_[MFC_OPTIN_DEVICES];   /* 0: not set yet; else 1 + cudaError_t of the opt-in */    \
        int dev_ = -1;                                                                                                \
        if (cudaGetDevice(&dev_) != cudaSuccess) return cudaErrorInvalidDevice;                                       \
        const bool cached_ = dev_ >= 0 && dev_ < MFC_OPTIN_DEVICES;                                                   \
        if (cached_) {                                                                                                \
            const int v_ = st_[dev_].load(std::memory_order_acquire);                                                 \
            if (v_) return (cudaError_t)(v_ - 1);                                                                     \
        }                                                                                                             \
        const cudaError_t e_ = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);      \
        if (cached_) st_[dev_].store(1 + (int)e_, std::memory_order_release);                                         \
        return e_;                                                                                                    \
    }()

// rank-4 tensor map (x, y, z, equation) of the padded state array with a box of bx x by cells of one plane, all equations
static bool encode_state_map(CUtensorMap *map, const Geo &g, int neq, const double *base, int bx, int by)
{
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn fn = []() -> encode_fn {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) != cudaSuccess || qr != cudaDriverEntryPointSuccess)
            return nullptr;
        return reinterpret_cast<encode_fn>(p);
    }();
    if (!fn) return false;
    // a map depends on the array's address, the padded extents and the box only: the last few are kept per host thread (an RK
    // step alternates between three arrays and two boxes), so a launch normally encodes nothing
    struct Key { const double *base; int p0, p1, p2, neq, bx, by; };
    struct Slot { Key k; CUtensorMap m; bool used; };
    static thread_local Slot cache[8] = {};
    static thread_local unsigned next = 0;
    const Key key{base, g.p[0], g.p[1], g.p[2], neq, bx, by};
    for (const Slot &sl : cache)
        if (sl.used && sl.k.base == key.base && sl.k.p0 == key.p0 && sl.k.p1 == key.p1 && sl.k.p2 == key.p2 && sl.k.neq == key.neq &&
            sl.k.bx == key.bx && sl.k.by == key.by) {
            *map = sl.m;
            return true;
        }
    const cuuint64_t dims[4] = {(cuuint64_t)g.p[0], (cuuint64_t)g.p[1], (cuuint64_t)g.p[2], (cuuint64_t)neq};
    const cuuint64_t strides[3] = {(cuuint64_t)g.sy * 8, (cuuint64_t)g.sz * 8, (cuuint64_t)g.cells * 8};
    const cuuint32_t box[4] = {(cuuint32_t)bx, (cuuint32_t)by, 1, (cuuint32_t)neq};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    if (fn(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<double *>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
           CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return false;
    Slot &sl = cache[next++ % 8];
    sl.k = key;
    sl.m = *map;
    sl.used = true;
    return true;
}

template <int D, int NF, int ORDER, bool NU>
static cudaError_t launch_fused_nu(const typename GeoOf<NU>::type &g, const Eos &e, const double *q, const SweepOut &o, int segment, int path, cudaStream_t s)
{
    constexpr int TY = fused_ty<D, NF>();
    using C = FusedCfg<D, NF, TY>;
    static_assert(C::bytes <= 227 * 1024, "fused tile does not fit shared memory");
    const int ntx = (g.n[0] + FTX - 1) / FTX;
    const int nty = D >= 2 ? (g.n[1] + TY - 1) / TY : 1;
    cudaError_t st;
    if constexpr (D == 3) {
        // one block per multiprocessor is what the TMEM allocation (all 512 columns) relies on
        static_assert(2 * C::bytes > 227 * 1024, "two resident blocks would deadlock in tcgen05.alloc");
        const int seg = fused_segment(g, (long long)ntx * nty, segment);
        const int nseg = (g.n[2] + seg - 1) / seg;
        const unsigned blocks = (unsigned)((long long)ntx * nty * nseg);
        // TMA staging needs 16-byte aligned rows (even padded extent, aligned base) and q_s = the array L is evaluated on
        using T = TmaCfg<NF, TY>;
        static_assert(T::bytes <= 227 * 1024, "TMA-staged tile does not fit shared memory");
        const bool tma_ok = path != MFC_PATH_LDGSTS && (g.p[0] & 1) == 0 && (reinterpret_cast<unsigned long long>(q) & 15) == 0 &&
                            (o.nbase == 0 || o.qs == q);
        CUtensorMap tm_plane, tm_col;
        // kernel with the z direction on specialised warps (mfc_fused_roles.cuh): the TMA layout conditions;
        // AUTO prefers it where it applies (256^3, two fluids: 2.31 against 2.55 ms per evaluation; 384^3, three: 9.9 against 11.7)
        {
            // (three fluids on a non-uniform grid: 464 B of spills in the split kernel; AUTO keeps the one-loop kernel there)
            if ((path == MFC_PATH_ROLES || (path == MFC_PATH_AUTO && (!NU || NF <= 2))) && tma_ok) {
                constexpr int RTY = MFC_ROLES_TY;
                using R = RolesCfg<NF, RTY>;
                const int rnty = (g.n[1] + RTY - 1) / RTY;
                const int rseg = fused_segment(g, (long long)ntx * rnty, segment, 1.0);
                const unsigned rblocks = (unsigned)((long long)ntx * rnty * ((g.n[2] + rseg - 1) / rseg));
                if (encode_state_map(&tm_plane, g, C::NEQ, q, FPX, RTY + 2 * NG) && encode_state_map(&tm_col, g, C::NEQ, q, R::CW, 1)) {
                    constexpr int rbytes = NU && R::nu_staged ? R::bytes_nu : R::bytes;
                    if ((st = MFC_OPTIN_SHARED((rhs_fused_roles_kernel<NF, RTY, ORDER, NU>), rbytes)) != cudaSuccess) return st;
                    rhs_fused_roles_kernel<NF, RTY, ORDER, NU><<<rblocks, R::THREADS, rbytes, s>>>(tm_plane, tm_col, g, e, o, ntx, rnty, rseg);
                    return cudaSuccess;
                }
            }
        }
        if (path == MFC_PATH_ROLES) return cudaErrorInvalidValue;
        if (tma_ok && encode_state_map(&tm_plane, g, C::NEQ, q, FPX, C::PY) && encode_state_map(&tm_col, g, C::NEQ, q, T::CW, TY)) {
            if ((st = MFC_OPTIN_SHARED((rhs_fused_march_tma_kernel<NF, TY, ORDER, NU>), T::bytes)) != cudaSuccess) return st;
            rhs_fused_march_tma_kernel<NF, TY, ORDER, NU><<<blocks, C::NT, T::bytes, s>>>(tm_plane, tm_col, g, e, o, ntx, nty, seg);
        } else {
            if (path == MFC_PATH_TMA) return cudaErrorInvalidValue;
            if ((st = MFC_OPTIN_SHARED((rhs_fused_march_kernel<NF, TY, ORDER, NU>), C::bytes)) != cudaSuccess) return st;
            rhs_fused_march_kernel<NF, TY, ORDER, NU><<<blocks, C::NT, C::bytes, s>>>(g, e, q, o, ntx, nty, seg);
        }
    } else {
        if ((st = MFC_OPTIN_SHARED((rhs_fused_plane_kernel<D, NF, TY, ORDER, NU>), C::bytes)) != cudaSuccess) return st;
        rhs_fused_plane_kernel<D, NF, TY, ORDER, NU><<<(unsigned)((long long)ntx * nty), C::NT, C::bytes, s>>>(g, e, q, o, ntx);
    }
    return cudaSuccess;
}

// non-uniform spacing (Geo::nonuniform) selects the table-driven instantiation; it exists for WENO5 only
template <int D, int NF, int ORDER>
static cudaError_t launch_fused(const GeoNu &g, const Eos &e, const double *q, const SweepOut &o, int segment, int path, cudaStream_t s)
{
    if (g.nu[0]) {
        if constexpr (ORDER == 5) return launch_fused_nu<D, NF, ORDER, true>(g, e, q, o, segment, path, s);
        else return cudaErrorInvalidValue;
    }
    return launch_fused_nu<D, NF, ORDER, false>(g, e, q, o, segment, path, s);
}

template <int D, int NF>
static cudaError_t launch_fused_order(int order, const GeoNu &g, const Eos &e, const double *q, const SweepOut &o, int segment, int path,
                                      cudaStream_t s)
{
    cudaError_t st = cudaSuccess;
    MFC_FOR_ORDER(order, (st = launch_fused<D, NF, ORDER>(g, e, q, o, segment, path, s)))
    return st;
}

cudaError_t MFC_CAT(launch_rhs_d, MFC_D)(int nf, int order, const GeoNu &g, const Eos &e, const double *q, const SweepOut &o,
                                         int segment, int path, cudaStream_t s)
{
    constexpr int D = MFC_D;
    cudaError_t err = cudaSuccess;
    MFC_FOR_NF(nf, (err = launch_fused_order<D, NF>(order, g, e, q, o, segment, path, s)))
    return err != cudaSuccess ? err : cudaGetLastError();
}

cudaError_t MFC_CAT(launch_cfl_d, MFC_D)(int nf, const GeoNu &g, const Eos &e, const double *q, unsigned long long *min_bits,
                                         cudaStream_t s)
{
    constexpr int D = MFC_D;
    const long long ncell = (long long)g.n[0] * g.n[1] * g.n[2];
    if (ncell >= (1ll << 32)) return cudaErrorInvalidValue;          // (the kernel indexes cells with 32 bits; 4 G cells do not fit a B200 anyway)
    long long want = (ncell + 255) / 256;
    const unsigned blocks = (unsigned)(want < 148 * 16 ? (want < 1 ? 1 : want) : 148 * 16);
    if (g.nu[0]) { MFC_FOR_NF(nf, (cfl_kernel<D, NF, true><<<blocks, 256, 0, s>>>(g, e, q, min_bits))) }
    else { MFC_FOR_NF(nf, (cfl_kernel<D, NF, false><<<blocks, 256, 0, s>>>((const Geo &)g, e, q, min_bits))) }
    return cudaGetLastError();
}

template <int D, int NF, int DIR>
static cudaError_t launch_line_t(int order, const Eos &e, int n, const double *w, double *vL, double *vR, double *F, double *uf,
                                 const double *nu, int nus, cudaStream_t s)
{
    if (nu) {
        if (order != 5) return cudaErrorInvalidValue;
        line_weno_kernel<D, NF, DIR, 5, true><<<(n + 2 + 127) / 128, 128, 0, s>>>(e, n, w, vL, vR, nu, nus);
    } else {
        MFC_FOR_ORDER(order, (line_weno_kernel<D, NF, DIR, ORDER, false><<<(n + 2 + 127) / 128, 128, 0, s>>>(e, n, w, vL, vR, nullptr, 0)))
    }
    line_hllc_kernel<D, NF, DIR><<<(n + 1 + 127) / 128, 128, 0, s>>>(e, n, vL, vR, F, uf);
    return cudaSuccess;
}

cudaError_t MFC_CAT(launch_line_d, MFC_D)(int nf, int order, int dir, const Eos &e, int n, const double *w, double *vL, double *vR,
                                          double *F, double *uf, const double *nu, int nus, cudaStream_t s)
{
    constexpr int D = MFC_D;
    if (dir < 0 || dir >= D) return cudaErrorInvalidValue;
    if (dir == 0) { MFC_FOR_NF(nf, (launch_line_t<D, NF, 0>(order, e, n, w, vL, vR, F, uf, nu, nus, s))) }
#if MFC_D >= 2
    else if (dir == 1) { MFC_FOR_NF(nf, (launch_line_t<D, NF, 1>(order, e, n, w, vL, vR, F, uf, nu, nus, s))) }
#endif
#if MFC_D >= 3
    else if (dir == 2) { MFC_FOR_NF(nf, (launch_line_t<D, NF, 2>(order, e, n, w, vL, vR, F, uf, nu, nus, s))) }
#endif
    return cudaGetLastError();
}

}  // namespace mfc
