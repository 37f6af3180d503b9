// The 3D right-hand side with the work of a tile split between SPECIALISED warps (uniform grid, two fluids):
// same decomposition as rhs_fused_march_tma_kernel (tile of 32 x TY cells in (x, y), march along z three planes ahead,
// TMA-staged planes, z window in tensor memory), but instead of TY warps that each run the whole per-plane schedule in
// lock step between block barriers, the block has one small loop per ROLE:
//   X warps  (TY / 2)  rows 2w, 2w + 1 of the staged plane: WENO + HLLC along x (exchange by shuffles), differences -> Lx
//                      (a buffer only this warp touches); then, one plane later, Lx + Ly + Lz, the Runge-Kutta combine and
//                      the one store of the cell (a4 + a5)
//   Y warps  (TY / 2)  the same rows along y: the face between the two rows is solved in registers, the right state of
//                      the lower row and the flux of the upper face go to the neighbouring warps through shared memory
//                      behind two barriers of the Y GROUP only (bar.sync with an id and a thread count) -> Ly
//   Z warps  (TY / 2)  columns of the same rows: raw row of plane m (TMA box) -> primitives -> ring of four planes in
//                      tensor memory; cell m - 2 reconstructed, face solved against the parked left state, difference
//                      -> Lz; own cells of plane m - 2 written into the staged plane
//   XR warp            rim of the tile in x (states of the cells -1 and 32, rim faces) + 7/10 of the halo cons->prim
//   YR warp            rim in y (states of the rows -1 and TY, rim faces)               + 3/10 of the halo cons->prim
// There is no producer warp: a Z warp re-issues the box of its own raw rows as soon as it has read them, and the LAST warp
// to finish with a staged plane (an atomic count) issues the box that overwrites it.
// The roles meet only through mbarriers (full / empty pairs per buffer, phases counted per plane; the L buffers pair the
// X, Y and Z warp of the same two rows), so a scheduler always holds warps in different phases of different loops: while
// the Y group waits at its barrier or a Z warp waits for tensor memory, X warps issue FP64.  Every loop is small enough
// for 96 registers per thread, which is what lets 20 warps (5 per scheduler) be resident instead of 12 (3 per scheduler)
// at 168 registers.  Roles are dealt to warp ids so that every scheduler (warp id mod 4) gets about the same FP64 work:
// (X, X, Y, Z, XR), (X, Y, Y, Z, YR), (X, X, Y, Z, Z), (X, Y, Y, Z, Z).
#pragma once
#include <cstdio>
#include "mfc_fused_tma.cuh"

namespace mfc {

__device__ __forceinline__ void mbar_arrive(unsigned long long *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_addr(bar)) : "memory");
}
// all lanes have finished their accesses (reads or writes) of the buffer the barrier guards; one arrival per warp
__device__ __forceinline__ void warp_arrive(unsigned long long *bar, int lane)
{
    __syncwarp();
    if (lane == 0) mbar_arrive(bar);
}
// wait with back-off: a warp that finds the phase incomplete sleeps instead of spinning on the issue port of a scheduler
// it shares with four working warps
__device__ __forceinline__ void mbar_wait_sleep(unsigned long long *bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra MFC_RDONE;\n"
        "MFC_RWAIT:\n"
        "nanosleep.u32 40;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@!p bra MFC_RWAIT;\n"
        "MFC_RDONE:\n"
        "}\n" ::"r"(smem_addr(bar)), "r"(parity)
        : "memory");
}
#ifdef MFC_ROLES_DEBUG
static __device__ __noinline__ void mbar_wait_dbg(unsigned long long *bar, unsigned parity, int line)
{
    for (long long it = 0; it < (1ll << 24); ++it) {
        unsigned ok;
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}\n" : "=r"(ok) : "r"(smem_addr(bar)), "r"(parity) : "memory");
        if (ok) return;
    }
    if ((threadIdx.x & 31) == 0) printf("STUCK block %d warp %d line %d parity %u\n", blockIdx.x, threadIdx.x >> 5, line, parity);
    __nanosleep(1000000);
    asm volatile("trap;");
}
#define RWAIT(bar, parity) mbar_wait_dbg(bar, parity, __LINE__)
#else
#define RWAIT(bar, parity) mbar_wait_sleep(bar, parity)
#endif
__device__ __forceinline__ void group_barrier(int id, int threads) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory"); }
__device__ __forceinline__ void fence_async_proxy() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// two doubles (4 columns) of the thread's own TMEM lane; the caller waits (tcgen05.wait::ld) once for a batch
__device__ __forceinline__ void tmem_load2_nowait(unsigned a, unsigned (&r)[4])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(a));
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ double pair_double(unsigned lo, unsigned hi) { return __hiloint2double((int)hi, (int)lo); }

#ifdef MFC_ROLES_CALL
// ONE copy of the reconstruction for all roles (a real call): the role loops together are larger than the instruction
// caches (L0 6 KB, L1.5 32 KB), and five different loops run on every scheduler at once
template <int ORDER>
static __device__ __noinline__ double2 reconstruct_call(double c, double dm2, double dm1, double d0, double d1, double eps4)
{
    double vL, vR;
    reconstruct<ORDER>(c, dm2, dm1, d0, d1, eps4, vL, vR);
    return make_double2(vL, vR);
}
template <int ORDER>
__device__ __forceinline__ void rc(double c, double dm2, double dm1, double d0, double d1, double eps4, double &vL, double &vR)
{
    const double2 v = reconstruct_call<ORDER>(c, dm2, dm1, d0, d1, eps4);
    vL = v.x;
    vR = v.y;
}
#else
template <int ORDER>
__device__ __forceinline__ void rc(double c, double dm2, double dm1, double d0, double d1, double eps4, double &vL, double &vR)
{
    reconstruct<ORDER>(c, dm2, dm1, d0, d1, eps4, vL, vR);
}
#endif

template <int NF, int TY>
struct RolesCfg {
    using C = FusedCfg<3, NF, TY>;
    static constexpr int NEQ = C::NEQ, NT = C::NT, PPL = C::PPL, NH = C::NH;
    static constexpr int RW = 2;                                         // rows per compute warp
    static constexpr int NW = TY / RW;                                   // warps per direction
    static constexpr int WARPS = 3 * NW + 2, THREADS = 32 * WARPS;
    static constexpr int PLANE_READERS = 2 * NW + 2;                     // X, Y, XR, YR warps
    // role of every warp id (see the file header): kind 0 X, 1 Y, 2 Z, 3 XR, 4 YR; index within the kind
    enum { K_X = 0, K_Y = 1, K_Z = 2, K_XR = 3, K_YR = 4 };
    static_assert(NW == 6, "the role table below is written for 6 + 6 + 6 + 2 warps");
    static constexpr unsigned long long pack3(const int (&a)[20])
    {
        unsigned long long v = 0;
        for (int i = 0; i < 20; ++i) v |= (unsigned long long)a[i] << (3 * i);
        return v;
    }
    static constexpr int kinds_[20] = {K_X, K_X, K_X, K_X, K_X, K_Y, K_X, K_Y, K_Y, K_Y, K_Y, K_Y, K_Z, K_Z, K_Z, K_Z, K_XR, K_YR, K_Z, K_Z};
    static constexpr int index_[20] = {0, 1, 2, 3, 4, 0, 5, 1, 2, 3, 4, 5, 0, 1, 2, 3, 0, 0, 4, 5};
    static constexpr unsigned long long KINDS = pack3(kinds_), INDEX = pack3(index_);
    __device__ static __forceinline__ int kind(int w) { return (int)((KINDS >> (3 * w)) & 7ull); }
    __device__ static __forceinline__ int index(int w) { return (int)((INDEX >> (3 * w)) & 7ull); }
    static constexpr int CW = FTX + 2;                                   // own-row box: cells -1 .. FTX of one row, all variables
    static constexpr int r16(int v) { return (v + 15) / 16 * 16; }       // 128-byte granules, in doubles
    static constexpr int nPb = r16(NEQ * PPL);                           // one staged plane with halo
    static constexpr int nSQr = r16(NEQ * CW);                           // raw own cells of one row of plane m: [NEQ][CW]
    static constexpr int oSQ = 2 * nPb;                                  // [TY] of them
    static constexpr int oYX = oSQ + TY * nSQr;                          // [NEQ][NW][32]     right state of every warp's lower row
    static constexpr int oYF = oYX + NEQ * NW * FTX;                     // [NEQ + 1][NW][32] flux + face velocity of every warp's upper face
    // x rim, per plane parity: HxR [NEQ][TY] (right state of the face past the tile), FxH [NEQ + 1][TY] (flux of face -1/2);
    // then XR's own scratch HxL, ExR [NEQ][TY] each (left and right state of face -1/2)
    static constexpr int nRXb = (2 * NEQ + 1) * TY;
    static constexpr int oRX = oYF + (NEQ + 1) * NW * FTX;
    // y rim, per plane parity: HyR [NEQ][32], FyH [NEQ + 1][32]; then YR's own scratch HyL [NEQ][32]
    static constexpr int nRYb = (2 * NEQ + 1) * FTX;
    static constexpr int oRY = oRX + 2 * nRXb + 2 * NEQ * TY;
    // flux differences of a plane, [NEQ][NT] each: Lx (written and read by the same thread, one plane apart), Ly, Lz[2]
    static constexpr int nL = NEQ * NT;
    static constexpr int oLx = r16(oRY + 2 * nRYb + NEQ * FTX);
    static constexpr int oLy = oLx + nL;
    static constexpr int oLz = oLy + nL;
    static constexpr int oBar = oLz + 2 * nL;
    // barriers (64-bit words at oBar)
    enum { FULL_P = 0, PRIM_P = 2, FULL_HXR = 4, FULL_FXH = 6, FULL_HYR = 8, FULL_FYH = 10, FULL_YX0 = 12,
           FULL_LY = 13, EMPTY_LY = FULL_LY + NW, FULL_LZ = EMPTY_LY + NW, EMPTY_LZ = FULL_LZ + 2 * NW,
           FULL_SQ = EMPTY_LZ + 2 * NW, NBAR = FULL_SQ + TY, TMEM_WORD = NBAR, CNT_P = NBAR + 1, NWORDS = NBAR + 2 };
    static constexpr int doubles = oBar + r16(NWORDS);
    static constexpr int bytes = doubles * (int)sizeof(double);
    static constexpr unsigned plane_bytes = NEQ * PPL * sizeof(double);
    static constexpr unsigned row_bytes = NEQ * CW * sizeof(double);
    // tensor memory of a Z thread, per row: ring of four primitive planes, parked left state, previous flux + face
    // velocity (2 TV columns each)
    static constexpr int TV = NEQ + 1 <= 8 ? 8 : 10;
    static constexpr int T_RING = 0, T_PARK = 4 * 2 * TV, T_FLUX = T_PARK + 2 * TV, T_ROW = T_FLUX + 2 * TV;
    static_assert(TV == 8, "the pairwise window loads below are written for 8 values per slot");
    static_assert(2 * RW * T_ROW <= 512, "TMEM columns (two Z warps per lane quarter)");
    static_assert(bytes <= 227 * 1024, "role-split tile does not fit shared memory");
    static_assert(2 * bytes > 227 * 1024, "two resident blocks would deadlock in tcgen05.alloc");
};

template <int NF, int TY, int ORDER>
__global__ void __launch_bounds__(RolesCfg<NF, TY>::THREADS, 1)
    rhs_fused_roles_kernel(const __grid_constant__ CUtensorMap tm_plane, const __grid_constant__ CUtensorMap tm_col, Geo g, Eos eos, SweepOut o,
                           int ntx, int nty, int seg)
{
    constexpr int D = 3;
    using R = RolesCfg<NF, TY>;
    using I = Idx<D, NF>;
    constexpr int NEQ = R::NEQ, NT = R::NT, PPL = R::PPL, NH = R::NH, NW = R::NW, CW = R::CW, TV = R::TV;
    extern __shared__ __align__(128) double sm[];
    double *const SQ = sm + R::oSQ;
    double *const YX = sm + R::oYX;
    double *const YF = sm + R::oYF;
    unsigned long long *const bars = reinterpret_cast<unsigned long long *>(sm + R::oBar);
    unsigned *const tmem_word = reinterpret_cast<unsigned *>(bars + R::TMEM_WORD);
    unsigned *const cnt_p = reinterpret_cast<unsigned *>(bars + R::CNT_P);   // [2] warps that are done with a staged plane

    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    const int kind = R::kind(warp), widx = R::index(warp);
    int bb = blockIdx.x;
    const int bx = bb % ntx;
    bb /= ntx;
    const int by = bb % nty, bs = bb / nty;
    const int x0 = bx * FTX, y0 = by * TY;
    const int k0 = bs * seg, k1 = min(k0 + seg, g.n[2]);
    const int U = k1 - k0;                                          // planes this block differences (u = 0 .. U - 1 is plane k0 + u)
    constexpr int POWN = NG * FPX + NG;                             // own cell (0, 0) of a staged plane

    if (tid == 0) {
        auto init = [&](int b, int n, unsigned count) { for (int k = 0; k < n; ++k) mbar_init(bars + b + k, count); };
        init(R::FULL_P, 2, 1);
        init(R::PRIM_P, 2, NW + 2);
        init(R::FULL_HXR, 2, 1);
        init(R::FULL_FXH, 2, 1);
        init(R::FULL_HYR, 2, 1);
        init(R::FULL_FYH, 2, 1);
        init(R::FULL_YX0, 1, 1);
        init(R::FULL_LY, NW, 1);
        init(R::EMPTY_LY, NW, 1);
        init(R::FULL_LZ, 2 * NW, 1);
        init(R::EMPTY_LZ, 2 * NW, 1);
        init(R::FULL_SQ, TY, 1);
        cnt_p[0] = 0;
        cnt_p[1] = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_async_proxy();
    }
    if (warp == 0) tmem_alloc512(tmem_word);
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const unsigned tmem_base = *tmem_word;

    // phase parity of the k-th use (k = 0, 1, ...) of a barrier
    auto par = [](int k) -> unsigned { return (unsigned)(k & 1); };
    // halo cell h (row-major numbering of the staged plane that skips the interior block) -> position in the plane
    auto halo_pos = [](int h) -> int {
        constexpr int TOP = NG * FPX;
        if (h < TOP) return h;
        if (h < TOP + 2 * NG * TY) {
            const int r = (h - TOP) / (2 * NG), k = (h - TOP) - r * 2 * NG;
            return (NG + r) * FPX + (k < NG ? k : FTX + k);
        }
        return (NG + TY) * FPX + (h - TOP - 2 * NG * TY);
    };
    // cons->prim in place of the halo cells h0 + lane, h0 + 32 + lane, ... < h1 of a landed plane
    auto convert_halo = [&](double *Pb, int h0, int h1) {
#pragma unroll 1
        for (int h = h0 + lane; h < h1; h += 32) {
            const int c = halo_pos(h);
            double qc[NEQ], wc[NEQ];
#pragma unroll
            for (int e = 0; e < NEQ; ++e) qc[e] = Pb[e * PPL + c];
            cons_to_prim_cell<D, NF>(qc, eos, wc);
#pragma unroll
            for (int e = 0; e < NEQ; ++e) Pb[e * PPL + c] = wc[e];
        }
    };
    constexpr int HSPLIT = ((NH * 7 / 10) + 31) / 32 * 32;          // halo cells below HSPLIT: XR, the rest: YR
    auto load_plane = [&](int v) {                                  // plane k0 + v with its halo -> P[v & 1] (one thread)
        mbar_expect_tx(bars + R::FULL_P + (v & 1), R::plane_bytes);
        tma_load_4d(sm + (v & 1) * R::nPb, &tm_plane, bars + R::FULL_P + (v & 1), x0, y0, k0 + v + NG, 0);
    };
    auto load_row = [&](int row, int n) {                           // raw cells of one row of plane k0 - 3 + n -> SQ[row] (one thread)
        mbar_expect_tx(bars + R::FULL_SQ + row, R::row_bytes);
        tma_load_4d(SQ + row * R::nSQr, &tm_col, bars + R::FULL_SQ + row, x0 + NG - 1, y0 + NG + row, k0 + n, 0);
    };
    // this warp is done with staged plane u; the last of the PLANE_READERS warps to say so issues the box of plane u + 2
    // into the same buffer (the count only grows: the k-th use of the buffer ends at (k + 1) PLANE_READERS)
    auto release_plane = [&](int u) {
        __syncwarp();
        if (lane == 0) {
            unsigned old;
            asm volatile("atom.acq_rel.cta.shared::cta.add.u32 %0, [%1], 1;" : "=r"(old) : "r"(smem_addr(cnt_p + (u & 1))) : "memory");
            if (old + 1 == (unsigned)(((u >> 1) + 1) * R::PLANE_READERS) && u + 2 < U) {
                fence_async_proxy();
                load_plane(u + 2);
            }
        }
    };
    if (tid == 0) {                                                 // both staged-plane buffers are free at the start
        load_plane(0);
        if (U > 1) load_plane(1);
    }

    if (kind == R::K_X) {
        // =====================================================  X  =====================================================
        const int xw = widx;
        double *const Lx = sm + R::oLx;
        const double *const Ly = sm + R::oLy;
        const double cx = o.coef * g.inv_dx[0], cy = o.coef * g.inv_dx[1], cz = o.coef * g.inv_dx[2];
#pragma unroll 1
        for (int u = 0; u <= U; ++u) {
            // ---- a4 + a5 for plane u - 1: out = ca q_n + cb q_s + coef (Lx / dx + Ly / dy + Lz / dz) ----
            if (u >= 1) {
                const int pu = u - 1;
                const double *const Lz = sm + R::oLz + (pu & 1) * R::nL;
                RWAIT(bars + R::FULL_LY + xw, par(pu));
                RWAIT(bars + R::FULL_LZ + 2 * xw + (pu & 1), par(pu >> 1));
#pragma unroll 1
                for (int r = 0; r < R::RW; ++r) {
                    const int row = R::RW * xw + r;
                    if (x0 + lane < g.n[0] && y0 + row < g.n[1]) {
                        const long long cell = (long long)(k0 + pu + NG) * g.sz + (long long)(y0 + row + NG) * g.sy + (x0 + lane + NG);
                        double qs[NEQ], qn[NEQ];
                        if (o.nbase > 0) {
#pragma unroll
                            for (int e = 0; e < NEQ; ++e) qs[e] = __ldcg(o.qs + (long long)e * g.cells + cell);
                        }
                        if (o.nbase > 1) {
#pragma unroll
                            for (int e = 0; e < NEQ; ++e) qn[e] = __ldcg(o.qn + (long long)e * g.cells + cell);
                        }
#pragma unroll
                        for (int e = 0; e < NEQ; ++e) {
                            const int c = e * NT + row * FTX + lane;
                            double a = fma(cx, Lx[c], fma(cy, Ly[c], cz * Lz[c]));
                            if (o.nbase > 0) a = fma(o.cb, qs[e], a);
                            if (o.nbase > 1) a = fma(o.ca, qn[e], a);
                            o.out[(long long)e * g.cells + cell] = a;
                        }
                    }
                }
                warp_arrive(bars + R::EMPTY_LY + xw, lane);
                warp_arrive(bars + R::EMPTY_LZ + 2 * xw + (pu & 1), lane);
            }
            if (u == U) break;
            // ---- x differences of plane u ----
            const int b = u & 1;
            const double *const Pb = sm + b * R::nPb;
            const double *const HxR = sm + R::oRX + b * R::nRXb;
            const double *const FxH = HxR + NEQ * TY;
            RWAIT(bars + R::PRIM_P + b, par(u >> 1));
#pragma unroll 1
            for (int r = 0; r < R::RW; ++r) {
                const int row = R::RW * xw + r;
                if (y0 + row >= g.n[1]) continue;                   // a row past the domain (ragged last tile): nothing reads its Lx
                if (o.nbase > 1 && x0 + lane < g.n[0] && u + 1 < U) {   // q_n of the next plane: into L2
                    const double *src = o.qn + (long long)(k0 + u + 1 + NG) * g.sz + (long long)(y0 + row + NG) * g.sy + (x0 + lane + NG);
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) prefetch_l2(src + (long long)e * g.cells);
                }
                const double *const pc = Pb + POWN + row * FPX + lane;
                double vL[NEQ], vR[NEQ];
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    const double *s5 = pc + e * PPL;
                    rc<ORDER>(s5[0], s5[-1] - s5[-2], s5[0] - s5[-1], s5[1] - s5[0], s5[2] - s5[1], eos.weno_eps4, vL[e], vR[e]);
                }
                RWAIT(bars + R::FULL_HXR + b, par(u >> 1));
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    const double nb = __shfl_down_sync(0xffffffffu, vR[e], 1);
                    vR[e] = lane == FTX - 1 ? HxR[e * TY + row] : nb;
                }
                double Fp[NEQ], ufp;
                hllc<D, NF, 0>(vL, vR, eos, Fp, ufp);
                RWAIT(bars + R::FULL_FXH + b, par(u >> 1));
                const double ufm = __shfl_up_sync(0xffffffffu, ufp, 1);
                const double du = ufp - (lane == 0 ? FxH[NEQ * TY + row] : ufm);
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    const double fm = __shfl_up_sync(0xffffffffu, Fp[e], 1);
                    double rr = (lane == 0 ? FxH[e * TY + row] : fm) - Fp[e];
                    if (e >= I::A) rr = fma(alpha_div_coef<NF>(eos, pc[e * PPL], pc[I::E * PPL]), du, rr);
                    Lx[e * NT + row * FTX + lane] = rr;
                }
            }
            release_plane(u);
        }
    } else if (kind == R::K_Y) {
        // =====================================================  Y  =====================================================
        const int yw = widx;
        const int ra = R::RW * yw, rb = ra + 1;                     // the warp's rows
        const bool skip = y0 + ra > g.n[1];                         // nothing of these rows reaches a cell of the domain
        double *const Ly = sm + R::oLy;
#pragma unroll 1
        for (int u = 0; u < U; ++u) {
            const int b = u & 1;
            const double *const Pb = sm + b * R::nPb;
            const double *const HyR = sm + R::oRY + b * R::nRYb;
            const double *const FyH = HyR + NEQ * FTX;
            RWAIT(bars + R::PRIM_P + b, par(u >> 1));
            const double *const pa = Pb + POWN + ra * FPX + lane;
            double Fi[NEQ], ui = 0.0, vLb[NEQ];
            if (!skip) {
                double vLa[NEQ], vRb[NEQ];
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    const double *s = pa + e * PPL;
                    const double dm2 = s[-FPX] - s[-2 * FPX], dm1 = s[0] - s[-FPX], d0 = s[FPX] - s[0], d1 = s[2 * FPX] - s[FPX], d2 = s[3 * FPX] - s[2 * FPX];
                    double vRa;
                    rc<ORDER>(s[0], dm2, dm1, d0, d1, eos.weno_eps4, vLa[e], vRa);
                    YX[(e * NW + yw) * FTX + lane] = vRa;
                    rc<ORDER>(s[FPX], dm1, d0, d1, d2, eos.weno_eps4, vLb[e], vRb[e]);
                }
                if (yw == 0) warp_arrive(bars + R::FULL_YX0, lane);
                hllc<D, NF, 1>(vLa, vRb, eos, Fi, ui);               // the face between the two rows
            } else if (yw == 0) {
                warp_arrive(bars + R::FULL_YX0, lane);
            }
            group_barrier(1, 32 * NW);                              // Y1: the right states of the lower rows are visible
            double ul = 0.0;
            if (!skip) {
                double vRn[NEQ], Fu[NEQ], uu;
                if (yw == NW - 1) RWAIT(bars + R::FULL_HYR + b, par(u >> 1));
#pragma unroll
                for (int e = 0; e < NEQ; ++e) vRn[e] = yw == NW - 1 ? HyR[e * FTX + lane] : YX[(e * NW + yw + 1) * FTX + lane];
                hllc<D, NF, 1>(vLb, vRn, eos, Fu, uu);               // the upper face
#pragma unroll
                for (int e = 0; e < NEQ; ++e) YF[(e * NW + yw) * FTX + lane] = Fu[e];
                YF[(NEQ * NW + yw) * FTX + lane] = uu;
                if (u >= 1) RWAIT(bars + R::EMPTY_LY + yw, par(u - 1));   // the X warp of these rows has combined plane u - 1
                const double du = uu - ui;
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    double rr = Fi[e] - Fu[e];
                    if (e >= I::A) rr = fma(alpha_div_coef<NF>(eos, pa[e * PPL + FPX], pa[I::E * PPL + FPX]), du, rr);
                    Ly[e * NT + rb * FTX + lane] = rr;
                }
            }
            group_barrier(2, 32 * NW);                              // Y2: the fluxes of the upper faces are visible
            if (!skip) {
                if (yw == 0) {
                    RWAIT(bars + R::FULL_FYH + b, par(u >> 1));
                    ul = FyH[NEQ * FTX + lane];
                } else {
                    ul = YF[(NEQ * NW + yw - 1) * FTX + lane];
                }
                const double du = ui - ul;
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    const double fl = yw == 0 ? FyH[e * FTX + lane] : YF[(e * NW + yw - 1) * FTX + lane];
                    double rr = fl - Fi[e];
                    if (e >= I::A) rr = fma(alpha_div_coef<NF>(eos, pa[e * PPL], pa[I::E * PPL]), du, rr);
                    Ly[e * NT + ra * FTX + lane] = rr;
                }
            }
            // (a warp that skips its rows still keeps step with the X warp of these rows: one phase of FULL_LY per plane)
            if (skip && u >= 1) RWAIT(bars + R::EMPTY_LY + yw, par(u - 1));
            warp_arrive(bars + R::FULL_LY + yw, lane);
            release_plane(u);
        }
    } else if (kind == R::K_Z) {
        // =====================================================  Z  =====================================================
        const int zw = widx;
        // lane quarter = warp id mod 4; the second Z warp of a quarter takes the upper half of the columns
        const unsigned tbase = tmem_base + ((unsigned)(32 * (warp & 3)) << 16) + (unsigned)(warp >= 16 ? 256 : 0);
        if (lane == 0) {
            for (int r = 0; r < R::RW; ++r) load_row(R::RW * zw + r, 0);
        }
#pragma unroll 1
        for (int n = 0; n < U + 2 * NG; ++n) {
            const int u = n - 2 * NG;                               // plane whose z difference is formed (if >= 0)
            const int v = n - 2 * NG + 1;                           // plane m - 2: reconstructed along z; own cells -> staged plane
            double *const Lz = sm + R::oLz + (u & 1) * R::nL;
            if (u >= 2) RWAIT(bars + R::EMPTY_LZ + 2 * zw + (u & 1), par((u - 2) >> 1));
#pragma unroll 1
            for (int r = 0; r < R::RW; ++r) {
                const int row = R::RW * zw + r;
                const unsigned trow = tbase + (unsigned)(r * R::T_ROW);
                double wn[TV];
                {
                    double qc[NEQ], w7[NEQ];
                    RWAIT(bars + R::FULL_SQ + row, par(n));
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) qc[e] = SQ[row * R::nSQr + e * CW + lane + 1];
                    __syncwarp();                                   // the raw row has been read: its box for the next plane
                    if (lane == 0 && n + 1 < U + 2 * NG) load_row(row, n + 1);
                    cons_to_prim_cell<D, NF>(qc, eos, w7);
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) wn[e] = w7[e];
#pragma unroll
                    for (int k = NEQ; k < TV; ++k) wn[k] = 0.0;
                }
                if (n >= 4) {
                    // window of the variables 2p, 2p + 1: planes m - 4 .. m - 1 from the ring (plane m - 4 sits in the slot
                    // plane m is about to take); reconstruct cell m - 2
                    double vLn[TV], vR[NEQ], vbE = 0.0, vbA[I::NA > 0 ? I::NA : 1];
#pragma unroll
                    for (int p = 0; p < TV / 2; ++p) {
                        unsigned w4[4], w3[4], w2[4], w1[4];
                        tmem_load2_nowait(trow + R::T_RING + (unsigned)(((n + 0) & 3) * 2 * TV + 4 * p), w4);
                        tmem_load2_nowait(trow + R::T_RING + (unsigned)(((n + 1) & 3) * 2 * TV + 4 * p), w3);
                        tmem_load2_nowait(trow + R::T_RING + (unsigned)(((n + 2) & 3) * 2 * TV + 4 * p), w2);
                        tmem_load2_nowait(trow + R::T_RING + (unsigned)(((n + 3) & 3) * 2 * TV + 4 * p), w1);
                        tmem_wait_ld();
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            const int e = 2 * p + h;
                            if (e < NEQ) {
                                const double a4 = pair_double(w4[2 * h], w4[2 * h + 1]), a3 = pair_double(w3[2 * h], w3[2 * h + 1]);
                                const double a2 = pair_double(w2[2 * h], w2[2 * h + 1]), a1 = pair_double(w1[2 * h], w1[2 * h + 1]);
                                rc<ORDER>(a2, a3 - a4, a2 - a3, a1 - a2, wn[e] - a1, eos.weno_eps4, vLn[e], vR[e]);
                                if (e == I::E) vbE = a3;
                                if (e >= I::A) vbA[e - I::A] = a3;
                            }
                        }
                    }
                    tmem_store<TV>(trow + R::T_RING + (unsigned)((n & 3) * 2 * TV), wn);
                    double vLp[TV];
                    tmem_load<TV>(trow + R::T_PARK, vLp);
#pragma unroll
                    for (int k = NEQ; k < TV; ++k) vLn[k] = 0.0;
                    tmem_store<TV>(trow + R::T_PARK, vLn);
                    if (n >= 5) {                                   // face (m - 2) - 1/2 lies in or on the edge of the segment
                        double Fp[NEQ], ufp, vl[NEQ];
#pragma unroll
                        for (int e = 0; e < NEQ; ++e) vl[e] = vLp[e];
                        hllc<D, NF, 2>(vl, vR, eos, Fp, ufp);
                        double Fm[TV], Fn[TV];
                        tmem_load<TV>(trow + R::T_FLUX, Fm);
#pragma unroll
                        for (int k = 0; k < TV; ++k) Fn[k] = 0.0;
#pragma unroll
                        for (int e = 0; e < NEQ; ++e) Fn[e] = Fp[e];
                        Fn[NEQ] = ufp;
                        tmem_store<TV>(trow + R::T_FLUX, Fn);
                        if (u >= 0) {
                            const double du = ufp - Fm[NEQ];
#pragma unroll
                            for (int e = 0; e < NEQ; ++e) {
                                double rr = Fm[e] - Fp[e];
                                if (e >= I::A) rr = fma(alpha_div_coef<NF>(eos, vbA[e - I::A], vbE), du, rr);
                                Lz[e * NT + row * FTX + lane] = rr;
                            }
                        }
                    }
                } else {
                    tmem_store<TV>(trow + R::T_RING + (unsigned)((n & 3) * 2 * TV), wn);
                }
            }
            if (u >= 0) warp_arrive(bars + R::FULL_LZ + 2 * zw + (u & 1), lane);
            // own cells of plane v (ring slot of plane m - 2) -> staged plane
            if (v >= 0 && v < U) {
                double *const Pb = sm + (v & 1) * R::nPb;
                RWAIT(bars + R::FULL_P + (v & 1), par(v >> 1));
#pragma unroll 1
                for (int r = 0; r < R::RW; ++r) {
                    const int row = R::RW * zw + r;
                    const unsigned trow = tbase + (unsigned)(r * R::T_ROW);
                    double w[TV];
                    tmem_load<TV>(trow + R::T_RING + (unsigned)(((n + 2) & 3) * 2 * TV), w);
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) Pb[e * PPL + POWN + row * FPX + lane] = w[e];
                }
                fence_async_proxy();                                // these writes precede the box that will overwrite the plane
                warp_arrive(bars + R::PRIM_P + (v & 1), lane);
            }
        }
    } else if (kind == R::K_XR) {
        // ================================  x rim + the first part of the halo conversion  ================================
        double *const HxL = sm + R::oRX + 2 * R::nRXb;              // [NEQ][TY] left state of face -1/2 (from cell -1)
        double *const ExR = HxL + NEQ * TY;                         // [NEQ][TY] right state of face -1/2 (from cell 0)
        RWAIT(bars + R::FULL_P, 0);
        convert_halo(sm, 0, HSPLIT);
        fence_async_proxy();
        warp_arrive(bars + R::PRIM_P, lane);
#pragma unroll 1
        for (int u = 0; u < U; ++u) {
            const int b = u & 1;
            const double *const Pb = sm + b * R::nPb;
            double *const HxR = sm + R::oRX + b * R::nRXb;
            double *const FxH = HxR + NEQ * TY;
            RWAIT(bars + R::PRIM_P + b, par(u >> 1));
            // units (kind, variable, row): kind 0 left state from cell -1, kind 1 right state from cell FTX, kind 2 right
            // state from cell 0.  A right state is the left state of the mirrored stencil
            constexpr int UX = 3 * TY * NEQ;
#pragma unroll 1
            for (int t = lane; t < UX; t += 32) {
                const int kd = t / (TY * NEQ), rem = t - kd * (TY * NEQ);
                const int e = rem / TY, r = rem - e * TY;
                const double *pb = Pb + e * PPL + POWN + r * FPX + (kd == 0 ? -1 : (kd == 1 ? FTX : 0));
                const int st = kd == 0 ? 1 : -1;
                double *dst = (kd == 0 ? HxL : (kd == 1 ? HxR : ExR)) + e * TY + r;
                double vv, other;
                rc<ORDER>(pb[0], pb[-st] - pb[-2 * st], pb[0] - pb[-st], pb[st] - pb[0], pb[2 * st] - pb[st], eos.weno_eps4, vv, other);
                *dst = vv;
            }
            warp_arrive(bars + R::FULL_HXR + b, lane);
            if (lane < TY) {
                double hl[NEQ], hr[NEQ], F[NEQ], uf;
#pragma unroll
                for (int e = 0; e < NEQ; ++e) { hl[e] = HxL[e * TY + lane]; hr[e] = ExR[e * TY + lane]; }
                hllc<D, NF, 0>(hl, hr, eos, F, uf);
#pragma unroll
                for (int e = 0; e < NEQ; ++e) FxH[e * TY + lane] = F[e];
                FxH[NEQ * TY + lane] = uf;
            }
            warp_arrive(bars + R::FULL_FXH + b, lane);
            release_plane(u);
            if (u + 1 < U) {
                RWAIT(bars + R::FULL_P + (b ^ 1), par((u + 1) >> 1));
                convert_halo(sm + (b ^ 1) * R::nPb, 0, HSPLIT);
                fence_async_proxy();
                warp_arrive(bars + R::PRIM_P + (b ^ 1), lane);
            }
        }
    } else {
        // ================================  y rim + the rest of the halo conversion  ================================
        double *const HyL = sm + R::oRY + 2 * R::nRYb;              // [NEQ][32] left state of face -1/2 (from row -1)
        RWAIT(bars + R::FULL_P, 0);
        convert_halo(sm, HSPLIT, NH);
        fence_async_proxy();
        warp_arrive(bars + R::PRIM_P, lane);
#pragma unroll 1
        for (int u = 0; u < U; ++u) {
            const int b = u & 1;
            const double *const Pb = sm + b * R::nPb;
            double *const HyR = sm + R::oRY + b * R::nRYb;
            double *const FyH = HyR + NEQ * FTX;
            RWAIT(bars + R::PRIM_P + b, par(u >> 1));
#pragma unroll 1
            for (int t = 0; t < 2 * NEQ; ++t) {                     // kind 0: left state from row -1; kind 1: right state from row TY
                const int kd = t / NEQ, e = t - kd * NEQ;
                const double *pb = Pb + e * PPL + POWN + (kd == 0 ? -1 : TY) * FPX + lane;
                const int st = kd == 0 ? FPX : -FPX;
                double vv, other;
                rc<ORDER>(pb[0], pb[-st] - pb[-2 * st], pb[0] - pb[-st], pb[st] - pb[0], pb[2 * st] - pb[st], eos.weno_eps4, vv, other);
                (kd == 0 ? HyL : HyR)[e * FTX + lane] = vv;
            }
            warp_arrive(bars + R::FULL_HYR + b, lane);
            RWAIT(bars + R::FULL_YX0, par(u));
            {
                double hl[NEQ], hr[NEQ], F[NEQ], uf;
#pragma unroll
                for (int e = 0; e < NEQ; ++e) { hl[e] = HyL[e * FTX + lane]; hr[e] = YX[(e * NW) * FTX + lane]; }
                hllc<D, NF, 1>(hl, hr, eos, F, uf);
#pragma unroll
                for (int e = 0; e < NEQ; ++e) FyH[e * FTX + lane] = F[e];
                FyH[NEQ * FTX + lane] = uf;
            }
            warp_arrive(bars + R::FULL_FYH + b, lane);
            release_plane(u);
            if (u + 1 < U) {
                RWAIT(bars + R::FULL_P + (b ^ 1), par((u + 1) >> 1));
                convert_halo(sm + (b ^ 1) * R::nPb, HSPLIT, NH);
                fence_async_proxy();
                warp_arrive(bars + R::PRIM_P + (b ^ 1), lane);
            }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) tmem_dealloc512(tmem_base);
}

}  // namespace mfc
