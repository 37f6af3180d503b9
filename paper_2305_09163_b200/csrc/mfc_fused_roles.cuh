// The 3D right-hand side with the work of a tile split between SPECIALISED warps (uniform grid, two fluids):
// same decomposition as rhs_fused_march_tma_kernel (tile of 32 x TY cells in (x, y), march along z three planes ahead,
// TMA-staged planes, z window in tensor memory), but instead of TY warps that each run the whole per-plane schedule in
// lock step between block barriers, the block has one small loop per ROLE:
//   X warps  (TY / 2)  rows 2w, 2w + 1 of the staged plane: WENO + HLLC along x (exchange by shuffles), differences -> Lx
//   Y warps  (TY / 2)  the same rows along y: the face between the two rows is solved in registers, the right state of
//                      the lower row and the flux of the upper face go to the neighbouring warps through shared memory
//                      behind two barriers of the Y GROUP only (bar.sync with an id and a thread count) -> Ly
//   Z warps  (TY / 2)  columns of the same rows: raw column of plane m (TMA box SQ) -> primitives -> z window (tensor
//                      memory, one slot of 4 planes per variable, shifted every plane), cell m - 2 reconstructed, face
//                      solved against the parked left state, difference -> Lz; own cells of plane m - 2 written into the
//                      staged plane; then Lx + Ly + Lz, the Runge-Kutta combine and the one store of cell m - 3
//   XR warp            rim of the tile in x (states of the cells -1 and 32, rim faces) + 7/10 of the halo cons->prim
//   YR warp            rim in y (states of the rows -1 and TY, rim faces)               + 3/10 of the halo cons->prim
// There is no producer warp: a Z warp re-issues the box of its own raw rows as soon as it has read them, and the LAST warp
// to finish with a staged plane (an atomic count) issues the box that overwrites it.
// The roles meet only through mbarriers (full / empty pairs per buffer, phases counted per plane), so a scheduler always
// holds warps in different phases of different loops: while the Y group waits at its barrier or a Z warp waits for
// tensor memory, X warps issue FP64.  Every loop is small enough for 96 registers per thread, which is what lets 20
// warps (5 per scheduler) be resident instead of 12 (3 per scheduler) at 168 registers.
// Work per plane is about equal for every warp (2 rows x (7 WENO + HLLC) = 960 FP64 instructions; XR and YR about 770).
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
#define RWAIT(bar, parity) mbar_wait(bar, parity)
#endif
__device__ __forceinline__ void group_barrier(int id, int threads) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory"); }
__device__ __forceinline__ void fence_async_proxy() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// four doubles (8 columns) of the thread's own TMEM lane
__device__ __forceinline__ void tmem_load4(unsigned a, double (&v)[4])
{
    unsigned r[8];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "r"(a));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int k = 0; k < 4; ++k) v[k] = __hiloint2double((int)r[2 * k + 1], (int)r[2 * k]);
}
__device__ __forceinline__ void tmem_store4(unsigned a, const double (&v)[4])
{
    unsigned r[8];
#pragma unroll
    for (int k = 0; k < 4; ++k) { r[2 * k] = (unsigned)__double2loint(v[k]); r[2 * k + 1] = (unsigned)__double2hiint(v[k]); }
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                 ::"r"(a), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]) : "memory");
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}

template <int NF, int TY>
struct RolesCfg {
    using C = FusedCfg<3, NF, TY>;
    static constexpr int NEQ = C::NEQ, NT = C::NT, PPL = C::PPL, NH = C::NH;
    static constexpr int RW = 2;                                         // rows per compute warp
    static constexpr int NW = TY / RW;                                   // warps per direction
    static constexpr int W_X = 0, W_Y = NW, W_Z = 2 * NW, W_XR = 3 * NW, W_YR = 3 * NW + 1;
    static constexpr int WARPS = 3 * NW + 2, THREADS = 32 * WARPS;
    static constexpr int PLANE_READERS = 2 * NW + 2;                     // X, Y, XR, YR warps
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
    static constexpr int nLb = 2 * NEQ * NT;                             // Lx [NEQ][NT], then Ly [NEQ][NT]
    static constexpr int oL = r16(oRY + 2 * nRYb + NEQ * FTX);           // two buffers (plane parity)
    static constexpr int oBar = oL + 2 * nLb;
    static constexpr int doubles = oBar + 48;
    static constexpr int bytes = doubles * (int)sizeof(double);
    static constexpr unsigned plane_bytes = NEQ * PPL * sizeof(double);
    static constexpr unsigned row_bytes = NEQ * CW * sizeof(double);
    // barriers (64-bit words at oBar)
    enum { FULL_P = 0, PRIM_P = 2, FULL_HXR = 4, FULL_FXH = 6, FULL_HYR = 8, FULL_FYH = 10, FULL_L = 12, EMPTY_L = 14, FULL_YX0 = 16,
           FULL_SQ = 17, NBAR = FULL_SQ + TY, TMEM_WORD = NBAR, CNT_P = NBAR + 1 };
    static_assert(CNT_P + 1 <= 48, "barrier words");
    // tensor memory of a Z thread, per row: NEQ windows of 4 planes (8 columns each), parked left state, previous flux +
    // face velocity, Lz of the cell waiting for Lx and Ly (2 TV columns each)
    static constexpr int TV = NEQ + 1 <= 8 ? 8 : 10;
    static constexpr int T_WIN = 0, T_PARK = 8 * NEQ, T_FLUX = T_PARK + 2 * TV, T_ACC = T_FLUX + 2 * TV, T_ROW = T_ACC + 2 * TV;
    static_assert(TY % RW == 0 && (W_Z & 3) == 0, "Z warps start at a multiple of four: warp & 3 is the TMEM lane quarter");
    static_assert(RW * T_ROW * ((NW + 3) / 4) <= 512, "TMEM columns");
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
        init(R::FULL_SQ, TY, 1);
        cnt_p[0] = 0;
        cnt_p[1] = 0;
        init(R::FULL_HXR, 2, 1);
        init(R::FULL_FXH, 2, 1);
        init(R::FULL_HYR, 2, 1);
        init(R::FULL_FYH, 2, 1);
        init(R::FULL_L, 2, 2 * NW);
        init(R::EMPTY_L, 2, NW);
        init(R::FULL_YX0, 1, 1);
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

    if (warp < R::W_Y) {
        // =====================================================  X  =====================================================
        const int xw = warp - R::W_X;
#pragma unroll 1
        for (int u = 0; u < U; ++u) {
            const int b = u & 1;
            const double *const Pb = sm + b * R::nPb;
            double *const Lx = sm + R::oL + b * R::nLb;
            const double *const HxR = sm + R::oRX + b * R::nRXb;
            const double *const FxH = HxR + NEQ * TY;
            RWAIT(bars + R::PRIM_P + b, par(u >> 1));
#pragma unroll 1
            for (int r = 0; r < R::RW; ++r) {
                const int row = R::RW * xw + r;
                if (y0 + row >= g.n[1]) continue;                   // a row past the domain (ragged last tile): nothing reads its Lx
                const double *const pc = Pb + POWN + row * FPX + lane;
                double vL[NEQ], vR[NEQ];
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    const double *s5 = pc + e * PPL;
                    reconstruct<ORDER>(s5[0], s5[-1] - s5[-2], s5[0] - s5[-1], s5[1] - s5[0], s5[2] - s5[1], eos.weno_eps4, vL[e], vR[e]);
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
                if (u >= 2) RWAIT(bars + R::EMPTY_L + b, par((u - 2) >> 1));
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    const double fm = __shfl_up_sync(0xffffffffu, Fp[e], 1);
                    double rr = (lane == 0 ? FxH[e * TY + row] : fm) - Fp[e];
                    if (e >= I::A) rr = fma(alpha_div_coef<NF>(eos, pc[e * PPL], pc[I::E * PPL]), du, rr);
                    Lx[e * NT + row * FTX + lane] = rr;
                }
            }
            warp_arrive(bars + R::FULL_L + b, lane);
            release_plane(u);
        }
    } else if (warp < R::W_Z) {
        // =====================================================  Y  =====================================================
        const int yw = warp - R::W_Y;
        const int ra = R::RW * yw, rb = ra + 1;                     // the warp's rows
        const bool skip = y0 + ra > g.n[1];                         // nothing of these rows reaches a cell of the domain
#pragma unroll 1
        for (int u = 0; u < U; ++u) {
            const int b = u & 1;
            const double *const Pb = sm + b * R::nPb;
            double *const Ly = sm + R::oL + b * R::nLb + NEQ * NT;
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
                    reconstruct<ORDER>(s[0], dm2, dm1, d0, d1, eos.weno_eps4, vLa[e], vRa);
                    YX[(e * NW + yw) * FTX + lane] = vRa;
                    reconstruct<ORDER>(s[FPX], dm1, d0, d1, d2, eos.weno_eps4, vLb[e], vRb[e]);
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
                if (u >= 2) RWAIT(bars + R::EMPTY_L + b, par((u - 2) >> 1));
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
            warp_arrive(bars + R::FULL_L + b, lane);
            release_plane(u);
        }
    } else if (warp < R::W_XR) {
        // =====================================================  Z  =====================================================
        const int zw = warp - R::W_Z;
        const unsigned tbase = tmem_base + ((unsigned)(32 * (warp & 3)) << 16) + (unsigned)((zw >> 2) * R::RW * R::T_ROW);
        const double cx = o.coef * g.inv_dx[0], cy = o.coef * g.inv_dx[1], cz = o.coef * g.inv_dx[2];
        if (lane == 0) {
            for (int r = 0; r < R::RW; ++r) load_row(R::RW * zw + r, 0);
        }
#pragma unroll 1
        for (int n = 0; n < U + 2 * NG; ++n) {
            const int u = n - 2 * NG;                               // plane whose cells are completed and written (if >= 0)
            const int v = n - 2 * NG + 1;                           // plane m - 2: reconstructed along z; own cells -> staged plane
#pragma unroll 1
            for (int r = 0; r < R::RW; ++r) {
                const int row = R::RW * zw + r;
                const unsigned trow = tbase + (unsigned)(r * R::T_ROW);
                double wn[NEQ];
                {
                    double qc[NEQ];
                    RWAIT(bars + R::FULL_SQ + row, par(n));
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) qc[e] = SQ[row * R::nSQr + e * CW + lane + 1];
                    __syncwarp();                                   // the raw row has been read: its box for the next plane
                    if (lane == 0 && n + 1 < U + 2 * NG) load_row(row, n + 1);
                    cons_to_prim_cell<D, NF>(qc, eos, wn);
                }
                // window of variable e: planes m - 4 .. m - 1; reconstruct cell m - 2; shift plane m in
                double vLn[TV], vR[NEQ], vbE = 0.0, vbA[I::NA > 0 ? I::NA : 1];
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    double w[4];
                    tmem_load4(trow + R::T_WIN + 8 * e, w);
                    vLn[e] = 0.0; vR[e] = 0.0;
                    if (n >= 4) reconstruct<ORDER>(w[2], w[1] - w[0], w[2] - w[1], w[3] - w[2], wn[e] - w[3], eos.weno_eps4, vLn[e], vR[e]);
                    if (e == I::E) vbE = w[1];
                    if (e >= I::A) vbA[e - I::A] = w[1];
                    const double ws[4] = {w[1], w[2], w[3], wn[e]};
                    tmem_store4(trow + R::T_WIN + 8 * e, ws);
                }
                if (n >= 4) {
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
                        const double du = ufp - Fm[NEQ];
                        double az[TV];
#pragma unroll
                        for (int k = NEQ; k < TV; ++k) az[k] = 0.0;
#pragma unroll
                        for (int e = 0; e < NEQ; ++e) {
                            double rr = Fm[e] - Fp[e];
                            if (e >= I::A) rr = fma(alpha_div_coef<NF>(eos, vbA[e - I::A], vbE), du, rr);
                            az[e] = cz * rr;                        // meaningful when u >= 0
                        }
                        tmem_store<TV>(trow + R::T_ACC, az);
                    }
                }
            }
            // own cells of plane v (now at position 1 of the shifted windows) -> staged plane; q_n of plane u + 1 -> L2
            if (v >= 0 && v < U) {
                double *const Pb = sm + (v & 1) * R::nPb;
                RWAIT(bars + R::FULL_P + (v & 1), par(v >> 1));
#pragma unroll 1
                for (int r = 0; r < R::RW; ++r) {
                    const int row = R::RW * zw + r;
                    const unsigned trow = tbase + (unsigned)(r * R::T_ROW);
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) {
                        double w[4];
                        tmem_load4(trow + R::T_WIN + 8 * e, w);
                        Pb[e * PPL + POWN + row * FPX + lane] = w[1];
                    }
                    if (o.nbase > 1 && x0 + lane < g.n[0] && y0 + row < g.n[1]) {
                        const double *src = o.qn + (long long)(k0 + v + NG) * g.sz + (long long)(y0 + row + NG) * g.sy + (x0 + lane + NG);
#pragma unroll
                        for (int e = 0; e < NEQ; ++e) prefetch_l2(src + (long long)e * g.cells);
                    }
                }
                fence_async_proxy();                                // these writes precede the box that will overwrite the plane
                warp_arrive(bars + R::PRIM_P + (v & 1), lane);
            }
            // a4 + a5: out = ca q_n + cb q_s + coef (Lx / dx + Ly / dy + Lz / dz)
            if (u >= 0) {
                const int b = u & 1;
                const double *const Lx = sm + R::oL + b * R::nLb;
                const double *const Ly = Lx + NEQ * NT;
                RWAIT(bars + R::FULL_L + b, par(u >> 1));
#pragma unroll 1
                for (int r = 0; r < R::RW; ++r) {
                    const int row = R::RW * zw + r;
                    const unsigned trow = tbase + (unsigned)(r * R::T_ROW);
                    double az[TV];
                    tmem_load<TV>(trow + R::T_ACC, az);             // (tcgen05.ld is warp-wide: outside the per-lane condition)
                    if (x0 + lane < g.n[0] && y0 + row < g.n[1]) {
                        const long long cell = (long long)(k0 + u + NG) * g.sz + (long long)(y0 + row + NG) * g.sy + (x0 + lane + NG);
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
                            double a = fma(cx, Lx[e * NT + row * FTX + lane], fma(cy, Ly[e * NT + row * FTX + lane], az[e]));
                            if (o.nbase > 0) a = fma(o.cb, qs[e], a);
                            if (o.nbase > 1) a = fma(o.ca, qn[e], a);
                            o.out[(long long)e * g.cells + cell] = a;
                        }
                    }
                }
                warp_arrive(bars + R::EMPTY_L + b, lane);
            }
        }
    } else if (warp == R::W_XR) {
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
                const int kind = t / (TY * NEQ), rem = t - kind * (TY * NEQ);
                const int e = rem / TY, r = rem - e * TY;
                const double *pb = Pb + e * PPL + POWN + r * FPX + (kind == 0 ? -1 : (kind == 1 ? FTX : 0));
                const int st = kind == 0 ? 1 : -1;
                double *dst = (kind == 0 ? HxL : (kind == 1 ? HxR : ExR)) + e * TY + r;
                double vv, other;
                reconstruct<ORDER>(pb[0], pb[-st] - pb[-2 * st], pb[0] - pb[-st], pb[st] - pb[0], pb[2 * st] - pb[st], eos.weno_eps4, vv, other);
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
                const int kind = t / NEQ, e = t - kind * NEQ;
                const double *pb = Pb + e * PPL + POWN + (kind == 0 ? -1 : TY) * FPX + lane;
                const int st = kind == 0 ? FPX : -FPX;
                double vv, other;
                reconstruct<ORDER>(pb[0], pb[-st] - pb[-2 * st], pb[0] - pb[-st], pb[st] - pb[0], pb[2 * st] - pb[st], eos.weno_eps4, vv, other);
                (kind == 0 ? HyL : HyR)[e * FTX + lane] = vv;
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
