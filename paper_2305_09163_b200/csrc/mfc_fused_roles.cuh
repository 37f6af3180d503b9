// The 3D right-hand side with the z direction split off to SPECIALISED warps (any number of fluids; uniform grid or per-index tables):
// same decomposition as rhs_fused_march_tma_kernel (tile of 32 x TY cells in (x, y), march along z three planes ahead,
// TMA-staged planes, z window in tensor memory), but the block has two kinds of warps, each with a loop of its own:
//   in-plane warps (TY, one row each): the x and y differences of the staged plane (inplane_xy, mfc_fused.cuh, its two
//       barriers now barriers of these warps only) and a4 + a5: Lx + Ly in registers + Lz from shared memory, the
//       Runge-Kutta combine and the one store of the cell;
//   Z warps (TY / ZR, ZR rows each): raw row of plane m (TMA box, re-issued by the warp as soon as it has read it) ->
//       primitives -> ring of four planes in tensor memory; cell m - 2 reconstructed, face solved against the parked left
//       state, difference -> Lz (shared memory, two buffers); own cells of plane m - 2 written into the staged plane,
//       whose halo cells (landed raw) they convert in place.
// The two kinds meet only through mbarriers (PRIM_P: own cells of a staged plane are primitives; FULL_LZ / EMPTY_LZ), so the
// z part -- a latency-bound chain (tensor-memory loads, one Riemann solve) that ran at half the FP64 rate when all warps
// of a scheduler were in it at once -- now overlaps the in-plane arithmetic of the other warps of its scheduler, and the
// in-plane loop no longer carries the z state in its registers.  16 warps, 128 registers, 4 per scheduler (3 + 1).
// (A finer split -- X, Y, Z, rim and conversion warps with five loops -- is in the history of this file: parity-exact but
// bound by instruction fetch: 85 KB of loop code per multiprocessor against a 32 KB instruction cache.)
#pragma once
#include <type_traits>
#include "mfc_fused_tma.cuh"

#ifndef MFC_ROLES_XPRE
#define MFC_ROLES_XPRE 4    // x reconstructions before barrier S1 (0 .. 7: 2.380 2.355 2.385 2.361 2.353 . . 2.414 ms at cfg3)
#endif

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
#define RWAIT(bar, parity) mbar_wait_sleep(bar, parity)
__device__ __forceinline__ void group_barrier(int id, int threads) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory"); }
__device__ __forceinline__ void fence_async_proxy() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// two doubles (4 columns) of the thread's own TMEM lane; the caller waits (tcgen05.wait::ld) once for a batch
__device__ __forceinline__ void tmem_load2_nowait(unsigned a, unsigned (&r)[4])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(a));
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ double pair_double(unsigned lo, unsigned hi) { return __hiloint2double((int)hi, (int)lo); }


template <int NF, int TY>
struct RolesCfg {
    using C = FusedCfg<3, NF, TY>;
    static constexpr int NEQ = C::NEQ, NT = C::NT, PPL = C::PPL, NH = C::NH, NHT = C::NHT;
    static constexpr int ZR = TY / 4;                                         // rows per Z warp
    static constexpr int NZ = TY / ZR;                                   // Z warps
    static constexpr int WARPS = TY + NZ, THREADS = 32 * WARPS;
    static constexpr int CW = FTX + 2;                                   // own-row box: cells -1 .. FTX of one row, all variables
    static constexpr int r16(int v) { return (v + 15) / 16 * 16; }       // 128-byte granules, in doubles
    static constexpr int nPb = r16(NEQ * PPL);                           // one staged plane with halo
    static constexpr int nSQr = r16(NEQ * CW);                           // raw own cells of one row of plane m: [NEQ][CW]
    static constexpr int oSQ = 2 * nPb;                                  // [TY] of them
    static constexpr int oRim = oSQ + TY * nSQr;                         // rim states and fluxes of inplane_xy
    static constexpr int oX8 = oRim + C::nHx + C::nHy;                   // y exchange: face velocity row
    static constexpr int oX = oX8 + NT;                                  //             right states [NEQ][NT]
    static constexpr int oX2 = oX + NEQ * NT;                            //             fluxes [NEQ][NT]
    static constexpr int nL = NEQ * NT;
    static constexpr int oLz = r16(oX2 + NEQ * NT);                      // z flux differences [2][NEQ][NT]
    static constexpr int NLZ = (TY > 12 || NEQ > 7) ? 1 : 2;               // (one buffer where two do not fit shared memory)
    static constexpr int oBar = oLz + NLZ * nL;
    enum { FULL_P = 0, PRIM_P = 2, FULL_LZ = 4, EMPTY_LZ = 6, FULL_SQ = 8, NBAR = FULL_SQ + TY, TMEM_WORD = NBAR, NWORDS = NBAR + 1 };
    static constexpr int doubles = oBar + r16(NWORDS);
    static constexpr int bytes = doubles * (int)sizeof(double);
    // non-uniform spacing only (after everything else): the block's slice of the coefficient tables as one record of NU_REC
    // doubles per cell (NuRec, mfc_math.cuh) -- columns -1 .. FTX of the x table, rows -1 .. TY of the y table -- and, per Z
    // warp, the record of the one cell along z its lanes are reconstructing
    static constexpr int oNuX = doubles, oNuY = oNuX + (FTX + 2) * NU_REC, oNuZ = oNuY + (TY + 2) * NU_REC;
    static constexpr int bytes_nu = (oNuZ + 4 * NU_REC) * (int)sizeof(double);
    static_assert(NU_REC % 2 == 0 && doubles % 2 == 0, "records are read with 16-byte loads");
    // (three fluids: the slices do not fit beside the tile; that instantiation keeps reading the tables from global memory)
    static constexpr bool nu_staged = bytes_nu <= 227 * 1024;
    static constexpr unsigned plane_bytes = NEQ * PPL * sizeof(double);
    static constexpr unsigned row_bytes = NEQ * CW * sizeof(double);
    // tensor memory of a Z thread, per row: ring of four primitive planes, parked left state, previous flux + face
    // velocity (2 TV columns each)
    static constexpr int TV = NEQ + 1 <= 8 ? 8 : 10;
    static constexpr int T_RING = 0, T_PARK = 4 * 2 * TV, T_FLUX = T_PARK + 2 * TV, T_ROW = T_FLUX + 2 * TV;
    static_assert(TY % ZR == 0 && NZ <= 4 && (TY & 3) == 0, "one Z warp per TMEM lane quarter (warp id mod 4)");
    static_assert(ZR * T_ROW <= 512, "TMEM columns");
    static_assert(bytes <= 227 * 1024, "tile does not fit shared memory");
    static_assert(2 * bytes > 227 * 1024, "two resident blocks would deadlock in tcgen05.alloc");
};

template <int NF, int TY, int ORDER, bool NU>
__global__ void __launch_bounds__(RolesCfg<NF, TY>::THREADS, 1)
    rhs_fused_roles_kernel(const __grid_constant__ CUtensorMap tm_plane, const __grid_constant__ CUtensorMap tm_col, typename GeoOf<NU>::type g, Eos eos,
                           SweepOut o, int ntx, int nty, int seg)
{
    constexpr int D = 3;
    using R = RolesCfg<NF, TY>;
    using C = FusedCfg<D, NF, TY>;
    using I = Idx<D, NF>;
    constexpr int NEQ = R::NEQ, NT = R::NT, PPL = R::PPL, NH = R::NH, CW = R::CW, TV = R::TV;
    extern __shared__ __align__(128) double sm[];
    double *const SQ = sm + R::oSQ;
    unsigned long long *const bars = reinterpret_cast<unsigned long long *>(sm + R::oBar);
    unsigned *const tmem_word = reinterpret_cast<unsigned *>(bars + R::TMEM_WORD);

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
        init(R::PRIM_P, 2, R::NZ);
        init(R::FULL_LZ, 2, R::NZ);
        init(R::EMPTY_LZ, 2, TY);
        init(R::FULL_SQ, TY, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_async_proxy();
    }
    constexpr bool NUSM = NU && R::nu_staged;                       // coefficient tables staged in shared memory
    if constexpr (NUSM) {
        // the tile's columns and rows do not change along the march: their coefficients come from global memory once
        // (rows of the tables are padded past the last cell, mfc_api.cu nu_tables: ragged tiles read defined entries)
        for (int t = tid; t < NU_NC * (FTX + 2 + TY + 2); t += R::THREADS) {
            const int k = t / (FTX + 2 + TY + 2), c = t - k * (FTX + 2 + TY + 2);
            if (c < FTX + 2) sm[R::oNuX + c * NU_REC + nu_rec_pos(k)] = __ldg(g.nu[0] + x0 + NG - 1 + c + k * g.nus[0]);
            else sm[R::oNuY + (c - FTX - 2) * NU_REC + nu_rec_pos(k)] = __ldg(g.nu[1] + y0 + NG - 1 + (c - FTX - 2) + k * g.nus[1]);
        }
    }
    if (warp == 0) tmem_alloc512(tmem_word);
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const unsigned tmem_base = *tmem_word;

    auto par = [](int k) -> unsigned { return (unsigned)(k & 1); };    // phase parity of the k-th use of a barrier
    auto lzb = [](int u) -> int { return R::NLZ == 2 ? (u & 1) : 0; };  // Lz buffer of plane u, and which use of it that is
    auto lzk = [](int u) -> int { return R::NLZ == 2 ? (u >> 1) : u; };
    auto load_plane = [&](int v) {                                  // plane k0 + v with its halo -> P[v & 1] (one thread)
        mbar_expect_tx(bars + R::FULL_P + (v & 1), R::plane_bytes);
        tma_load_4d(sm + (v & 1) * R::nPb, &tm_plane, bars + R::FULL_P + (v & 1), x0, y0, k0 + v + NG, 0);
    };
    auto load_row = [&](int row, int n) {                           // raw cells of one row of plane k0 - 3 + n -> SQ[row] (one thread)
        mbar_expect_tx(bars + R::FULL_SQ + row, R::row_bytes);
        tma_load_4d(SQ + row * R::nSQr, &tm_col, bars + R::FULL_SQ + row, x0 + NG - 1, y0 + NG + row, k0 + n, 0);
    };

    const double cz = o.coef * g.inv_dx[2];

    if (warp < TY) {
        // =================================================  in-plane warps  =================================================
        const int i = lane, j = warp;
        const bool active = x0 + i < g.n[0] && y0 + j < g.n[1];
        const long long col = (long long)(y0 + j + NG) * g.sy + (x0 + i + NG);
        if (tid == 0) {                                             // both staged-plane buffers are free at the start
            load_plane(0);
            if (U > 1) load_plane(1);
        }
        const InplaneBufs<D, NF, TY> B0(sm, sm + R::oRim, sm + R::oX, sm + R::oX2, sm + R::oX8);
        const InplaneBufs<D, NF, TY> B1(sm + R::nPb, sm + R::oRim, sm + R::oX, sm + R::oX2, sm + R::oX8);
#pragma unroll 1
        for (int u = 0; u < U; ++u) {
            const int b = u & 1;
            const long long cell = (long long)(k0 + u + NG) * g.sz + col;
            double coef = o.coef;
            asm volatile("" : "+d"(coef));
            double cx = coef * g.inv_dx[0], cy = coef * g.inv_dx[1], czp = cz;
            if constexpr (NU) {                                     // the cell's own widths (Eq. 8-9): entry 27 of the tables
                if constexpr (NUSM) {
                    cx = coef * sm[R::oNuX + (1 + i) * NU_REC + nu_rec_pos(27)];
                    cy = coef * sm[R::oNuY + (1 + j) * NU_REC + nu_rec_pos(27)];
                } else {
                    cx = coef * __ldg(g.nu[0] + x0 + NG + i + 27 * g.nus[0]);
                    cy = coef * __ldg(g.nu[1] + y0 + NG + j + 27 * g.nus[1]);
                }
                czp = coef * __ldg(g.nu[2] + k0 + u + NG + 27 * g.nus[2]);
            }
            RWAIT(bars + R::PRIM_P + b, par(u >> 1));                  // the Z warps have made plane u primitives (own cells and halo)
            double acc[NEQ];
#pragma unroll
            for (int e = 0; e < NEQ; ++e) acc[e] = 0.0;
            auto early = [&]() {                                    // q_n of the next plane: into L2
                if (active && o.nbase > 1 && u + 1 < U) {
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) prefetch_l2(o.qn + (long long)e * g.cells + cell + g.sz);
                }
            };
            if constexpr (NUSM) {                                   // per-index coefficient tables of the tile's columns and rows
                inplane_xy<D, NF, TY, ORDER, true, NT, MFC_ROLES_XPRE>(b ? B1 : B0, eos, cx, cy, acc, early, NoHook(),
                                                                       NuPlaneShared{smem_addr(sm + R::oNuX + NU_REC), smem_addr(sm + R::oNuY + NU_REC)});
            } else if constexpr (NU) {
                inplane_xy<D, NF, TY, ORDER, true, NT, MFC_ROLES_XPRE>(b ? B1 : B0, eos, cx, cy, acc, early, NoHook(),
                                                                       NuPlane{g.nu[0] + x0 + NG, g.nu[1] + y0 + NG, g.nus[0], g.nus[1]});
            } else {
                inplane_xy<D, NF, TY, ORDER, false, NT, MFC_ROLES_XPRE>(b ? B1 : B0, eos, cx, cy, acc, early, NoHook());
            }
            // ---- bottom: q_s (L2: this block read the cell as a raw row three planes ago) and q_n loaded now, used last ----
            double qsv[NEQ], qnv[NEQ];
            if (active) {
                if (o.nbase > 0) {
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) qsv[e] = __ldcg(o.qs + (long long)e * g.cells + cell);
                }
                if (o.nbase > 1) {
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) qnv[e] = __ldcg(o.qn + (long long)e * g.cells + cell);
                }
            }
            // ---- a4 + a5: out = ca q_n + cb q_s + coef (Lx / dx + Ly / dy + Lz / dz) ----
            RWAIT(bars + R::FULL_LZ + lzb(u), par(lzk(u)));
            {
                const double *const Lz = sm + R::oLz + lzb(u) * R::nL;
#pragma unroll
                for (int e = 0; e < NEQ; ++e) acc[e] = fma(czp, Lz[e * NT + tid], acc[e]);
            }
            warp_arrive(bars + R::EMPTY_LZ + lzb(u), lane);
            if (active) {
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    double a = acc[e];
                    if (o.nbase > 0) a = fma(o.cb, qsv[e], a);
                    if (o.nbase > 1) a = fma(o.ca, qnv[e], a);
                    o.out[(long long)e * g.cells + cell] = a;
                }
            }
            inplane_sync<NT>();                                     // plane u has been read by everybody
            if (tid == 0 && u + 2 < U) load_plane(u + 2);
        }
    } else {
        // =====================================================  Z warps  =====================================================
        const int zw = warp - TY;
        const unsigned tbase = tmem_base + ((unsigned)(32 * (warp & 3)) << 16);     // lane quarter = warp id mod 4
        if (lane == 0) {
            for (int r = 0; r < R::ZR; ++r) load_row(R::ZR * zw + r, 0);
        }
#pragma unroll 1
        for (int n = 0; n < U + 2 * NG; ++n) {
            const int u = n - 2 * NG;                               // plane whose z difference is formed (if >= 0)
            const int v = n - 2 * NG + 1;                           // plane m - 2: reconstructed along z; own cells -> staged plane
            double *const Lz = sm + R::oLz + lzb(u) * R::nL;
            if (u >= R::NLZ) RWAIT(bars + R::EMPTY_LZ + lzb(u), par(lzk(u - R::NLZ)));
            if constexpr (NUSM) {
                // the coefficients of cell m - 2 = k0 + v along z are the same for every thread and row: one load per lane,
                // then read back by all lanes (the warp's own 32 doubles of shared memory)
                if (n >= 4) {
                    __syncwarp();
                    if (lane < NU_NC) sm[R::oNuZ + NU_REC * zw + nu_rec_pos(lane)] = __ldg(g.nu[2] + k0 + v + NG + lane * g.nus[2]);
                    __syncwarp();
                }
            }
#pragma unroll 1
            for (int r = 0; r < R::ZR; ++r) {
                const int row = R::ZR * zw + r;
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
                    // tables of cell m - 2 = k0 + v (NU only)
                    const typename std::conditional<NUSM, NuRec, NuRef>::type nz = [&]() {
                        if constexpr (NUSM) return NuRec{smem_addr(sm + R::oNuZ + NU_REC * zw)};
                        else if constexpr (NU) return NuRef{g.nu[2] + k0 + v + NG, g.nus[2]};
                        else return NuRef{nullptr, 0};
                    }();
#pragma unroll
                    for (int p = 0; p < (NEQ + 1) / 2; ++p) {
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
                                reconstruct<ORDER, NU>(a2, a3 - a4, a2 - a3, a1 - a2, wn[e] - a1, eos.weno_eps4, vLn[e], vR[e], nz);
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
            if (u >= 0) warp_arrive(bars + R::FULL_LZ + lzb(u), lane);
            // own cells of plane v (ring slot of plane m - 2) -> staged plane
            if (v >= 0 && v < U) {
                double *const Pb = sm + (v & 1) * R::nPb;
                RWAIT(bars + R::FULL_P + (v & 1), par(v >> 1));
#pragma unroll 1
                for (int r = 0; r < R::ZR; ++r) {
                    const int row = R::ZR * zw + r;
                    const unsigned trow = tbase + (unsigned)(r * R::T_ROW);
                    double w[TV];
                    tmem_load<TV>(trow + R::T_RING + (unsigned)(((n + 2) & 3) * 2 * TV), w);
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) Pb[e * PPL + POWN + row * FPX + lane] = w[e];
                }
                // halo cells of the landed plane: raw q -> primitives in place, dealt to the Z warps in rounds of 32
#pragma unroll 1
                for (int h = 32 * zw + lane; h < NH; h += 32 * R::NZ) {
                    constexpr int TOP = NG * FPX;                   // (row-major numbering of the staged plane that skips the interior block)
                    int c;
                    if (h < TOP) c = h;
                    else if (h < TOP + 2 * NG * TY) {
                        const int rr = (h - TOP) / (2 * NG), kk = (h - TOP) - rr * 2 * NG;
                        c = (NG + rr) * FPX + (kk < NG ? kk : FTX + kk);
                    } else c = (NG + TY) * FPX + (h - TOP - 2 * NG * TY);
                    double qc[NEQ], wc[NEQ];
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) qc[e] = Pb[e * PPL + c];
                    cons_to_prim_cell<D, NF>(qc, eos, wc);
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) Pb[e * PPL + c] = wc[e];
                }
                fence_async_proxy();                                // these writes precede the box that will overwrite the plane
                warp_arrive(bars + R::PRIM_P + (v & 1), lane);
            }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) tmem_dealloc512(tmem_base);
}

}  // namespace mfc
